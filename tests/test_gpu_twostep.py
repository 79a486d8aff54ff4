"""GPU parity of the paper's own two-step form and of thermal emission in
the ray step (NEXT-3; eq. 8, App. A with source terms): the CUDA path through the C ABI against the oracle on the same
seeded inputs and packet ids.

Tolerances: the source grid is summed with fp32 reductions in arbitrary order from fp32 segment
integrals (3-point Gauss-Legendre for the U, V parts): per cell and camera |dS| <= 5e-5 x the cell's deposited I + 2e-6 x
the largest cell.  The ray step is fp64 on both sides: maps from the same source agree to 1e-9; maps of the whole
pipeline inherit the grid's tolerance.
"""
import math

import numpy as np
import pytest

from paper_2512_01283_b200 import inputs
from harness import (oracle_model, oracle_observers, gpu_grid, gpu_observers, gpu_events_sorted, compare_sequences, show)
from oracle import OracleEvents, OracleStats

pytestmark = pytest.mark.gpu


def _worst(img_g, img_o, floor_rel):
    """largest |difference| per pixel in units of that pixel's I (plus floor_rel x the brightest pixel)"""
    I = np.abs(img_o[:, :1])
    return float((np.abs(img_g - img_o) / (I + floor_rel * I.max())).max())

CASES = {
    "c1": dict(n=16, n_packets=20000, npix=32),        # scalar cells, Rayleigh
    "c2": dict(n=24, n_packets=8000, npix=32),         # scalar cells, HG table with S34
    "c4": dict(n=20, n_packets=6000, npix=32),         # general cells, helical field, volume source, 3 cameras
    "c5": dict(n=16, n_packets=3000, npix=24),         # general cells, random field, 8 cameras
}


def _oracle_two_step(cfg, n, npix, emis=None):
    m = oracle_model(cfg)
    obs = oracle_observers(cfg)
    ev = OracleEvents(max(1024, 40 * n)); st = OracleStats()
    sg, _, nseg = m.transport_deposit(0, n, cfg["seed"], ev, obs, stats=st)
    img, _ = m.image_rays(sg, obs, npix, npix, emis=emis)
    k = ev.n
    order = np.lexsort((ev.k[:k], ev.id[:k]))
    evd = dict(id=ev.id[:k][order], k=ev.k[:k][order], cell=ev.cell[:k][order], pos=ev.p[:k][order], dir=ev.n_in[:k][order],
               stokes=ev.S[:k][order])
    return m, sg.reshape(cfg["nz"], cfg["ny"], cfg["nx"], len(obs), 4), nseg, img, evd, st


def _non_cubic(name):
    """13 x 7 x 21 cells of 0.1 x 0.05 x 0.07 in an off-centre box, random density with empty cells (and random field): none of the
    BASELINE workloads has non-cubic cells or odd, unequal dimensions."""
    nx, ny, nz = 13, 7, 21
    rng = np.random.default_rng(78)
    cfg = inputs.make(name, n=8, n_packets=4000, npix=24)
    dens = np.exp(rng.uniform(math.log(0.05), math.log(30.0), size=(nz, ny, nx))).astype(np.float32)
    dens[rng.uniform(size=dens.shape) < 0.15] = 0.0
    bf = None if cfg["bfield"] is None else rng.normal(size=(nz, ny, nx, 3)).astype(np.float32)
    obs = [dict(theta=math.radians(t), phi=math.radians(f), center=[0.15, 0.275, -0.265], half_w=hw, half_h=hh)
           for t, f, hw, hh in ((0, 0, 0.8, 0.5), (57, 33, 0.9, 0.9), (141, 200, 0.7, 1.1))]
    src = dict(kind=0 if cfg["bfield"] is None else 1, pos=[0.11, 0.31, -0.4], dir=[0, 0, 1], cell_weight=None)
    return dict(cfg, nx=nx, ny=ny, nz=nz, bounds=[-0.5, 0.8, 0.1, 0.45, -1.0, 0.47], density=dens, bfield=bf, source=src, observers=obs)


@pytest.mark.parametrize("name", sorted(CASES) + ["c2-13x7x21", "c4-13x7x21"])
def test_source_grid_and_ray_image_against_the_oracle(name):
    cfg = _non_cubic(name[:2]) if "-" in name else inputs.make(name, **CASES[name])
    n, npix = cfg["n_packets"], cfg["npix"]
    m, sg_o, nseg_o, img_o, ev_o, st_o = _oracle_two_step(cfg, n, npix)
    obs = gpu_observers(cfg)
    # events without a source grid ...
    g0 = gpu_grid(cfg)
    g0.transport(n, cfg["seed"])
    ev_plain = gpu_events_sorted(g0)
    g0.close()
    # ... and with one: the same packets, the same events
    g = gpu_grid(cfg)
    g.sgrid_begin(obs)
    g.transport(n, cfg["seed"])
    ev_g = gpu_events_sorted(g)
    for key in ev_g:
        assert np.array_equal(ev_g[key], ev_plain[key]), key
    frac, info = compare_sequences(ev_o, ev_g, np.arange(n))
    assert frac >= 0.999, show(info)
    st = g.stats_get()
    assert abs(st["segments"] - nseg_o) <= 2e-3 * nseg_o + 2, (st["segments"], nseg_o)
    sg_g = g.sgrid_get().astype(np.float64)
    assert sg_g.shape == sg_o.shape
    # take the cells out that a disagreeing packet's path may touch (none at these sizes when frac == 1)
    ref = np.abs(sg_o[..., :1])
    tol = 5e-5 * ref + 2e-6 * ref.max()
    bad = np.abs(sg_g - sg_o) > tol
    if frac == 1.0:
        assert bad.sum() == 0, (name, int(bad.sum()), float((np.abs(sg_g - sg_o) / (ref + 1e-3 * ref.max())).max()))
    else:
        assert bad.sum() <= 40 * (1 - frac) * n * 30, (name, int(bad.sum()))
    assert abs(sg_g[..., 0].sum() / sg_o[..., 0].sum() - 1) < 1e-5
    # step 2 on the GPU's own grid against the oracle's pipeline
    g.image_rays(obs, npix, npix)
    img_g = g.image_get()
    assert _worst(img_g, img_o, 1e-2) < 1e-4, _worst(img_g, img_o, 1e-2)
    for s in range(4):
        assert abs(img_g[:, s].sum() - img_o[:, s].sum()) <= 2e-5 * img_o[:, 0].sum()
    # a second batch accumulates; reset clears
    g.sgrid_reset()
    assert not g.sgrid_get().any()
    g.sgrid_end()
    from paper_2512_01283_b200 import krp
    with pytest.raises(krp.KrpError) as ei:       # no open grid any more
        g.sgrid_get()
    assert ei.value.code == krp.ERR_STATE
    g.close()


def test_ray_step_alone_is_fp64_exact_and_adds_thermal_emission():
    """Step 2 from a source grid that holds only what one small transport left (GPU grid read back and handed to the
    oracle's ray step), with and without a thermal source: both sides fp64, maps agree to 1e-9; thermal emission alone
    needs no source grid."""
    cfg = inputs.make("c4", n=16, n_packets=3000, npix=40)
    for o in cfg["observers"]:
        o["center"] = [0.0123, -0.0077, 0.0051]      # no pixel ray of the axis-aligned views runs exactly along a cell face
    obs = gpu_observers(cfg)
    g = gpu_grid(cfg)
    g.sgrid_begin(obs)
    g.transport(cfg["n_packets"], cfg["seed"])
    sg = g.sgrid_get()
    rng = np.random.default_rng(5)
    emis = (0.3 * rng.uniform(0.5, 1.5, size=cfg["density"].shape)).astype(np.float32)
    m = oracle_model(cfg)
    oo = oracle_observers(cfg)
    for em in (None, emis):
        g.image_reset()
        g.image_rays(obs, 40, 28, emis=em)
        img_g = g.image_get()
        img_o, st = m.image_rays(sg.astype(np.float64).reshape(-1, len(oo), 4), oo, 40, 28, emis=em)
        assert _worst(img_g, img_o, 1e-3) < 1e-9, _worst(img_g, img_o, 1e-3)
    g.sgrid_end()
    import torch
    g.image_reset(); g.stats_reset()
    g.image_rays(obs, 40, 28, emis=torch.from_numpy(emis).cuda())          # device array, no source grid
    img_g = g.image_get()
    img_o, st = m.image_rays(None, oo, 40, 28, emis=emis)
    assert _worst(img_g, img_o, 1e-3) < 1e-9, _worst(img_g, img_o, 1e-3)
    stg = g.stats_get()
    assert stg["steps_image"] == st.steps_image and stg["contributions"] == st.contributions
    from paper_2512_01283_b200 import krp
    with pytest.raises(krp.KrpError) as ei:
        g.image_rays(obs, 8, 8)                                             # neither a grid nor a thermal source
    assert ei.value.code == krp.ERR_STATE
    g.sgrid_begin(obs[:2])
    with pytest.raises(krp.KrpError) as ei:
        g.image_rays(obs, 8, 8, emis=emis)                                  # not the grid's cameras
    assert ei.value.code == krp.ERR_ARG
    with pytest.raises(krp.KrpError):
        g.sgrid_begin(obs * 9)                                              # more than 16 cameras
    g.close()


def test_eq15_on_the_gpu():
    """PAPER.md:198 eq. 15 through the CUDA ray step: isothermal aligned slab, no scattering, up to tau = 30."""
    from paper_2512_01283_b200 import krp
    a1, a2 = 1.0, float(np.float32(0.12))
    p0 = a2 / a1
    for tau in (0.01, 1.0, 10.0, 30.0):
        tau = float(np.float32(tau))
        for n in (1, 33):
            dens = np.full((1, 1, n), tau, np.float32)
            bf = np.broadcast_to(np.array([0, 0, 1], np.float32), (1, 1, n, 3)).copy()
            opac = np.tile(np.array([a1, a2, 0.0, 0.0], np.float32), (2, 1))
            mu = np.tile(np.array([1.0, 0.0, 0.0, 0.0], np.float32), (5, 1))
            g = krp.Grid(n, 1, 1, [0, 1, 0, 1, 0, 1], dens, bf, mu, opac)
            o = [krp.make_observer(math.pi / 2, 0.0, [0.5, 0.5, 0.5], 0.5)]
            g.image_rays(o, 1, 1, emis=np.full((1, 1, n), 2.5, np.float32))
            I, Q, U, V = g.image_get()[0, :, 0, 0]
            P = math.exp(-tau) * math.sinh(p0 * tau) / (1 - math.exp(-tau) * math.cosh(p0 * tau))
            assert abs(I - 2.5 * (1 - math.exp(-tau) * math.cosh(p0 * tau))) < 1e-11 * 2.5
            assert abs(Q / I - P) < 1e-10 and abs(U) < 1e-13 and abs(V) < 1e-13
            g.close()


def test_two_step_image_matches_event_image_statistically():
    """On the GPU alone, at a size the oracle cannot reach: the paper's form and the per-event form of the same packets
    give the same image-integrated Stokes parameters within the discretisation of the grid form (cells of optical depth
    <= 0.1, pixel rays finer than cells) -- C4 at 64^3, 2^20 packets."""
    cfg = inputs.make("c4", n=64, n_packets=1 << 20, npix=256)
    obs = gpu_observers(cfg)
    g = gpu_grid(cfg)
    g.sgrid_begin(obs)
    g.events_reserve(6 << 20)
    g.transport(cfg["n_packets"], cfg["seed"])
    g.image(obs, 256, 256)
    img_e = g.image_get().copy()
    g.image_reset()
    g.image_rays(obs, 256, 256)
    img_r = g.image_get()
    for o in range(len(obs)):
        Ie, Ir = img_e[o, 0].sum(), img_r[o, 0].sum()
        assert abs(Ir / Ie - 1) < 0.02, (o, Ir, Ie)
        for s in (1, 2):
            assert abs(img_r[o, s].sum() - img_e[o, s].sum()) < 0.01 * Ie, (o, s)
    g.close()


def test_thermal_packet_source_matches_the_oracle():
    """Source kind 5 (reading R22): thermal emission of aligned grains as the packet source -- directions by rejection against
    (1 - omega) alpha1(mu), initial Stokes (1, alpha2/alpha1, 0, 0) in the grain frame -- event by event against the oracle,
    with a strongly direction-dependent table so that rejections are common; on a model with 4-byte cells it is the plain
    volume source."""
    from harness import oracle_run, compare_images_same_ids
    cfg = inputs.make("c4", n=16, n_packets=6000, npix=24)
    mu = np.linspace(0, 1, 9); s2 = 1 - mu * mu
    cfg["opacity"] = np.stack([1 + 0.3 * s2, 0.3 * s2, 0.1 * s2, 0.3 + 0.4 * mu], 1).astype(np.float32)
    cfg["source"] = dict(kind=5, pos=[0, 0, 0], dir=[0, 0, 1], cell_weight=np.ascontiguousarray(cfg["density"], np.float32))
    n = cfg["n_packets"]
    ora, img_o, img2_o, st_o = oracle_run(cfg, 0, n, cap=64 * n)
    g = gpu_grid(cfg)
    g.events_reserve(64 * n)
    g.transport(n, cfg["seed"])
    gev = gpu_events_sorted(g)
    frac, info = compare_sequences(ora, gev, np.arange(n))
    assert frac >= 0.999, show(info)
    first = ora["k"] == 1
    assert np.abs(ora["stokes"][first, 1:3]).max() > 0.05                     # the first events do carry the emitted polarisation
    g.image(gpu_observers(cfg), cfg["npix"], cfg["npix"])
    compare_images_same_ids(cfg, ora, gev, info, np.arange(n), g.image_get(), img_o, img2_o, cfg["npix"], cfg["npix"], name="thermal-source")
    g.close()
    from paper_2512_01283_b200 import krp
    with pytest.raises(krp.KrpError):
        gpu_grid(dict(cfg, source=dict(cfg["source"], kind=6)))               # thermal needs the volume source, isotropic candidates
    c1 = inputs.make("c1", n=12, n_packets=3000, npix=16)
    ev = {}
    for kind in (1, 5):
        c1["source"] = dict(kind=kind, pos=[0, 0, 0], dir=[0, 0, 1], cell_weight=None)
        g = gpu_grid(c1)
        g.transport(3000, 4)
        ev[kind] = gpu_events_sorted(g)
        g.close()
    for key in ev[1]:
        assert np.array_equal(ev[1][key], ev[5][key]), key
