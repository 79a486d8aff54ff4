"""Seeded synthetic workloads shaped like BASELINE.json's five configs.

This module holds NONE of the method's arithmetic: it only fills arrays (densities, field
directions, lookup tables) and lists sources and observers.  Both the CUDA tests/bench and the
oracle tests take their inputs from here; neither implementation imports the other.

All generation is numpy on the host (the same arrays reach both implementations); only the 3-D
FFT of the Gaussian random fields goes through torch for speed.
"""
import math

import numpy as np

N_ANG = 181
N_INC = 91


# ------------------------------------------------------------------------------------------
# tables
# ------------------------------------------------------------------------------------------
def rayleigh_mueller(n_ang=N_ANG):
    """Rayleigh phase matrix on the table nodes, (1/2) int S11 sin = 1."""
    c = np.cos(np.linspace(0.0, math.pi, n_ang))
    return np.stack([0.75 * (1 + c * c), -0.75 * (1 - c * c), 1.5 * c, np.zeros_like(c)], 1).astype(np.float32)


def hg_mueller(g=0.5, pmax=0.4, seed=0, n_ang=N_ANG, ripple=0.05, circ=0.2):
    """Smooth HG-like table: S11 = HG(g) x seeded ripple (<= ~5 %), normalised with the trapezoid rule;
    S12 = -pmax S11 sin^2/(1+cos^2); S33 = S11 2cos/(1+cos^2); S34 = -circ S11 sin^2/(1+cos^2)."""
    th = np.linspace(0.0, math.pi, n_ang)
    c, s = np.cos(th), np.sin(th)
    s11 = (1 - g * g) / (1 + g * g - 2 * g * c) ** 1.5
    a = np.random.default_rng(seed).normal(size=4)
    s11 = s11 * np.exp(ripple * sum(a[m - 1] * np.cos(m * th) for m in range(1, 5)) / 2.0)
    f = s11 * s
    norm = 0.5 * float(np.sum(0.5 * (f[1:] + f[:-1])) * (th[1] - th[0]))
    s11 = s11 / norm
    x = s * s / (1 + c * c)
    y = 2 * c / (1 + c * c)
    return np.stack([s11, -pmax * s11 * x, s11 * y, -circ * s11 * x], 1).astype(np.float32)


def constant_opacity(a1=1.0, albedo=0.5):
    return np.array([[a1, 0.0, 0.0, albedo]], np.float32)


def aligned_opacity(ratio=1.1, circ=0.02, albedo=0.5, n_inc=N_INC):
    """Aligned-grain set (reading R8) on mu = |cos vartheta| nodes: with s2 = 1 - mu^2,
    alpha1 = 1 + (R-1)/2 s2, alpha2 = (R-1)/2 s2, alpha3 = circ s2."""
    mu = np.linspace(0.0, 1.0, n_inc)
    s2 = 1.0 - mu * mu
    h = 0.5 * (ratio - 1.0)
    return np.stack([1 + h * s2, h * s2, circ * s2, np.full_like(mu, albedo)], 1).astype(np.float32)


def dipole_ztable(n_ti=37, n_to=37, n_dp=72, a_par=1.0, a_perp=1.0):
    """Synthetic full scattering matrix of aligned grains: an induced dipole with polarizability
    a_par along the grain axis (z of the grain frame) and a_perp across it (complex numbers allowed), Z[n_ti, n_to, n_dp, 4, 4]
    on incidence angle, outgoing polar angle and azimuth difference, Stokes vectors referenced to (theta^, phi^) of each
    direction in the grain frame (eq. 4-5), normalised so that the isotropic case is the Rayleigh matrix with mean(Z11) = 1.
    A stand-in for the paper's dipole-approximation grain model, whose formulas are not in the paper's text."""
    ti = np.radians(np.linspace(0.0, 180.0, n_ti))[:, None, None]
    to = np.radians(np.linspace(0.0, 180.0, n_to))[None, :, None]
    dp = np.radians(np.arange(n_dp) * 360.0 / n_dp)[None, None, :]
    one = np.ones(np.broadcast_shapes(ti.shape, to.shape, dp.shape))
    A = np.array([a_perp, a_perp, a_par], complex)
    thi = np.stack([np.cos(ti) * one, 0 * one, -np.sin(ti) * one], -1)
    phi = np.stack([0 * one, one, 0 * one], -1)
    tho = np.stack([np.cos(to) * np.cos(dp) * one, np.cos(to) * np.sin(dp) * one, -np.sin(to) * one], -1)
    pho = np.stack([-np.sin(dp) * one, np.cos(dp) * one, 0 * one], -1)
    J = np.empty(one.shape + (2, 2), complex)
    for r, eo in enumerate((tho, pho)):
        for c, ei in enumerate((thi, phi)):
            J[..., r, c] = (eo * A * ei).sum(-1)
    # Mueller matrix of a Jones matrix: M = T (J kron J*) T^-1, coherency vector (tt*, tp*, pt*, pp*), V = i (tp* - pt*)
    T = np.array([[1, 0, 0, 1], [1, 0, 0, -1], [0, 1, 1, 0], [0, 1j, -1j, 0]], complex)
    K = np.einsum("...ab,...cd->...acbd", J, J.conj()).reshape(one.shape + (4, 4))
    M = np.einsum("ij,...jk,kl->...il", T, K, np.linalg.inv(T)).real
    return (1.5 * M).astype(np.float32)


# ------------------------------------------------------------------------------------------
# fields
# ------------------------------------------------------------------------------------------
def _centres(n, lo, hi):
    d = (hi - lo) / n
    return lo + (np.arange(n) + 0.5) * d


def gaussian_random_field(n, seed, slope=-11.0 / 3.0):
    """Zero-mean, unit-variance Gaussian random field on an n^3 periodic grid with P(k) ~ k^slope."""
    import torch
    rng = np.random.default_rng(seed)
    noise = rng.standard_normal((n, n, n), dtype=np.float32)
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    t = torch.from_numpy(noise).to(dev)
    f = torch.fft.rfftn(t)
    k1 = torch.fft.fftfreq(n, 1.0 / n, device=dev)
    kz = torch.fft.rfftfreq(n, 1.0 / n, device=dev)
    k2 = k1[:, None, None] ** 2 + k1[None, :, None] ** 2 + kz[None, None, :] ** 2
    amp = torch.where(k2 > 0, k2.clamp_min(1e-30) ** (slope / 4.0), torch.zeros_like(k2))
    f = f * amp
    out = torch.fft.irfftn(f, s=(n, n, n))
    out = out - out.mean()
    out = out / out.std()
    return out.float().cpu().numpy()


# ------------------------------------------------------------------------------------------
# the five configs
# ------------------------------------------------------------------------------------------
def _observer(theta_deg, phi_deg, centre, half):
    return dict(theta=math.radians(theta_deg), phi=math.radians(phi_deg), center=list(centre), half_w=half, half_h=half)


def _base(name, n, bounds, density, bfield, mueller, opacity, source, observers, npix, n_packets, seed,
          w_min=1e-4, max_scatter=64):
    nx, ny, nz = n
    return dict(name=name, nx=nx, ny=ny, nz=nz, bounds=list(bounds),
                density=np.ascontiguousarray(density, np.float32),
                bfield=None if bfield is None else np.ascontiguousarray(bfield, np.float32),
                mueller=mueller, opacity=opacity, source=source, observers=observers,
                npix=npix, n_packets=int(n_packets), seed=int(seed), w_min=w_min, max_scatter=max_scatter)


def c1_uniform_sphere(n=32, n_packets=10 ** 5, npix=64):
    """C1: n^3 cells, kappa*rho constant inside r < L/2 (cell centres) with radial tau = 1, albedo 0.5, Rayleigh,
    isotropic point source at the centre, one observer at 60 deg inclination."""
    L = 1.0
    x = _centres(n, -L / 2, L / 2)
    r2 = x[None, None, :] ** 2 + x[None, :, None] ** 2 + x[:, None, None] ** 2
    dens = np.where(r2 < (L / 2) ** 2, 2.0 / L, 0.0)
    src = dict(kind=0, pos=[0.0, 0.0, 0.0], dir=[0, 0, 1], cell_weight=None)
    return _base("C1 uniform sphere %d^3" % n, (n, n, n), [-L / 2, L / 2] * 3, dens, None, rayleigh_mueller(),
                 constant_opacity(1.0, 0.5), src, [_observer(60, 0, (0, 0, 0), L / 2)], npix, n_packets, 1)


def c2_flared_disk(n=128, n_packets=10 ** 8, npix=256):
    """C2: rho ~ r^-1 exp(-z^2/2h^2), h = 0.1 r^1.25 (r, z, h in units of the grid radius), inner hole of
    2 cells, midplane tau = 20 from the centre to the edge; HG-like table g = 0.5, pmax = 0.4; 4 inclinations."""
    L = 1.0
    x = _centres(n, -1.0, 1.0)            # units of the grid radius L/2
    rc = np.sqrt(x[None, None, :] ** 2 + x[None, :, None] ** 2) + 0 * x[:, None, None]
    z = x[:, None, None] + 0 * rc
    h = 0.1 * np.maximum(rc, 1e-6) ** 1.25
    rho = np.where(rc >= 2 * (2.0 / n), np.exp(-0.5 * (z / h) ** 2) / np.maximum(rc, 1e-6), 0.0)
    rho = np.where(rc <= 1.0, rho, 0.0)
    row = rho[n // 2, n // 2, n // 2:]
    rho = rho * (20.0 / (row.sum() * (L / n)))
    src = dict(kind=0, pos=[0.0, 0.0, 0.0], dir=[0, 0, 1], cell_weight=None)
    obs = [_observer(t, 0, (0, 0, 0), L / 2) for t in (0, 30, 60, 85)]
    return _base("C2 flared disk %d^3" % n, (n, n, n), [-L / 2, L / 2] * 3, rho, None, hg_mueller(0.5, 0.4, seed=1002),
                 constant_opacity(1.0, 0.5), src, obs, npix, n_packets, 2)


def c3_aligned_slab(n=64, nz_factor=4, n_packets=10 ** 8, npix=128):
    """C3: n x n x 4n cubic cells, per-cell kappa*rho*dz log-uniform in [1e-3, 1e3] (R16), uniform B at 45 deg to z
    in the x-z plane, aligned set R = 1.1, c = 0.02, sources uniform in the volume, observer along +z."""
    nz = n * nz_factor
    dz = 1.0 / nz
    rng = np.random.default_rng(1003)
    tau_cell = np.exp(rng.uniform(math.log(1e-3), math.log(1e3), size=(nz, n, n)))
    dens = tau_cell / dz
    b = np.broadcast_to(np.array([math.sin(math.pi / 4), 0.0, math.cos(math.pi / 4)], np.float32), (nz, n, n, 3))
    w = n * dz
    src = dict(kind=1, pos=[w / 2, w / 2, 0.5], dir=[0, 0, 1], cell_weight=None)
    obs = [_observer(0, 0, (w / 2, w / 2, 0.5), w / 2)]
    return _base("C3 aligned slab %dx%dx%d" % (n, n, nz), (n, n, nz), [0, w, 0, w, 0, 1.0], dens, b,
                 hg_mueller(0.3, 0.4, seed=1003), aligned_opacity(1.1, 0.02, 0.5), src, obs, npix, n_packets, 3)


def c4_twisted_cylinder(n=256, n_packets=10 ** 9, npix=256):
    """C4: Gaussian radial density (sigma = 0.2 L) about the z axis with axial tau = 10, helical field
    B_phi/B_z = r/(0.1 L), aligned tables, volume source weighted by the density, three views."""
    L = 1.0
    x = _centres(n, -L / 2, L / 2)
    X = x[None, None, :] + np.zeros((n, n, n), np.float32)
    Y = x[None, :, None] + np.zeros((n, n, n), np.float32)
    r2 = X * X + Y * Y
    dens = (10.0 / L) * np.exp(-r2 / (2 * (0.2 * L) ** 2))
    b = np.stack([-Y / (0.1 * L), X / (0.1 * L), np.ones_like(X)], -1)
    src = dict(kind=1, pos=[0, 0, 0], dir=[0, 0, 1], cell_weight=np.ascontiguousarray(dens, np.float32))
    obs = [_observer(0, 0, (0, 0, 0), 0.7 * L), _observer(90, 0, (0, 0, 0), 0.7 * L), _observer(45, 30, (0, 0, 0), 0.7 * L)]
    return _base("C4 twisted cylinder %d^3" % n, (n, n, n), [-L / 2, L / 2] * 3, dens, b, hg_mueller(0.3, 0.4, seed=1004),
                 aligned_opacity(1.1, 0.02, 0.5), src, obs, npix, n_packets, 4)


def c5_turbulent_cloud(n=512, n_packets=10 ** 9, npix=512):
    """C5: lognormal density exp(g), g a Gaussian random field with P(k) ~ k^-11/3 and sigma = 1.5, mean tau = 5
    from the centre to a face; unit B from three independent fields of the same spectrum; albedo 0.6; 8 observers
    along the cube diagonals."""
    L = 1.0
    sig = 1.5
    g = gaussian_random_field(n, 1005)
    dens = np.exp(sig * g - 0.5 * sig * sig)
    dens *= 5.0 / (float(dens.mean(dtype=np.float64)) * (L / 2))
    b = np.stack([gaussian_random_field(n, 2005 + 10 * a) for a in range(3)], -1)
    src = dict(kind=0, pos=[0.0, 0.0, 0.0], dir=[0, 0, 1], cell_weight=None)
    t = math.degrees(math.acos(1 / math.sqrt(3)))
    obs = [_observer(th, ph, (0, 0, 0), math.sqrt(3) * L / 2) for th in (t, 180 - t) for ph in (45, 135, 225, 315)]
    return _base("C5 turbulent cloud %d^3" % n, (n, n, n), [-L / 2, L / 2] * 3, dens, b, hg_mueller(0.3, 0.4, seed=1005),
                 aligned_opacity(1.1, 0.02, 0.6), src, obs, npix, n_packets, 5)


CONFIGS = {"c1": c1_uniform_sphere, "c2": c2_flared_disk, "c3": c3_aligned_slab,
           "c4": c4_twisted_cylinder, "c5": c5_turbulent_cloud}


def make(name, **kw):
    """Build config `name` ("c1".."c5"); keyword arguments shrink it (n=, n_packets=, npix=)."""
    return CONFIGS[name](**kw)
