"""GPU parity with periodic boundaries (reading R20): the CUDA path against
the oracle, event by event and map by map, plus the closed forms the oracle is pinned to, run through the CUDA path."""
import math

import numpy as np
import pytest

from paper_2512_01283_b200 import inputs
from harness import (oracle_run, oracle_model, oracle_observers, gpu_grid, gpu_observers, gpu_events_sorted, compare_sequences,
                     compare_images_same_ids, show)

pytestmark = pytest.mark.gpu


def _cfg(mask, dichroic, shape=None):
    cfg = inputs.make("c4" if dichroic else "c1", n=12, n_packets=6000, npix=24)
    rng = np.random.default_rng(17)
    n = 12
    nx, ny, nz = shape or (n, n, n)
    if shape:      # non-cubic cells, odd unequal dimensions (0.1 x 0.14 x 0.05), box still centred on the observers' centre
        cfg.update(nx=nx, ny=ny, nz=nz, bounds=[-0.65, 0.65, -0.49, 0.49, -0.525, 0.525])
    cfg["density"] = (1.5 * np.exp(0.6 * rng.normal(size=(nz, ny, nx)))).astype(np.float32)          # no empty rim: packets do reach the faces
    if dichroic:
        cfg["bfield"] = rng.normal(size=(nz, ny, nx, 3)).astype(np.float32)
        cfg["source"] = dict(kind=1, pos=[0, 0, 0], dir=[0, 0, 1], cell_weight=None)
    else:
        cfg["source"] = dict(kind=0, pos=[0.31, -0.22, 0.05], dir=[0, 0, 1], cell_weight=None)
    cfg["observers"] = [dict(theta=math.radians(t), phi=math.radians(p), center=[0.0, 0.0, 0.0], half_w=1.2, half_h=1.2)
                        for t, p in ((10, 15), (35, 20), (70, 250))]      # no ray exactly parallel to an open face
    cfg["periodic"] = mask
    return cfg


@pytest.mark.parametrize("mask,dichroic,shape", [(3, False, None), (3, True, None), (5, True, None), (1, False, None),
                                                 (6, True, (13, 7, 21)), (2, False, (13, 7, 21))])
def test_periodic_sequences_and_images(mask, dichroic, shape):
    cfg = _cfg(mask, dichroic, shape)
    n = cfg["n_packets"]
    ora, img_o, img2_o, st_o = oracle_run(cfg, 0, n, cap=64 * n)
    g = gpu_grid(cfg)
    g.events_reserve(64 * n)
    g.transport(n, cfg["seed"])
    gev = gpu_events_sorted(g)
    frac, info = compare_sequences(ora, gev, np.arange(n))
    print("periodic", mask, dichroic, frac, show(info))
    assert frac >= 0.999, show(info)
    g.image(gpu_observers(cfg), cfg["npix"], cfg["npix"])
    img_g = g.image_get()
    st = g.stats_get()
    compare_images_same_ids(cfg, ora, gev, info, np.arange(n), img_g, img_o, img2_o, cfg["npix"], cfg["npix"], name="periodic")
    assert abs(st["steps_transport"] - st_o["steps_transport"]) <= 2e-3 * st_o["steps_transport"]
    # (an imaging ray stops once its attenuation is exactly 0 in fp32, so the kernel may take fewer steps than the oracle)
    assert st["steps_image"] <= st_o["steps_image"] * (1 + 2e-3) + 2 and st["steps_image"] >= 0.5 * st_o["steps_image"]
    # the open box is a different problem: more escapes
    cfg0 = dict(cfg, periodic=0)
    g0 = gpu_grid(cfg0)
    g0.transport(n, cfg["seed"])
    assert g0.stats_get()["w_escaped"] > st["w_escaped"] * 1.02
    # the same run with the per-observer arrays off (the march that does its own look-ups)
    g.tune_schedule(obs_cells=0)
    g.image_reset(); g.packet_id_set(0)
    g.transport(n, cfg["seed"])
    g.image(gpu_observers(cfg), cfg["npix"], cfg["npix"])
    img2 = g.image_get()
    assert np.abs(img2 - img_g).max() <= 2e-5 * np.abs(img_g[:, 0]).max()
    g.close(); g0.close()


def test_infinite_slab_escape_fraction_E2():
    """scipy.special.expn(2, tau): the closed form the oracle's periodic transport is pinned to, through the CUDA path."""
    import scipy.special
    from paper_2512_01283_b200 import krp
    tau, N = 1.5, 1 << 20
    dens = np.full((8, 8, 8), 2 * tau, np.float32)
    mu = np.tile(np.array([1.0, 0.0, 0.0, 0.0], np.float32), (5, 1))
    g = krp.Grid(8, 8, 8, [0, 1, 0, 1, 0, 1], dens, None, mu, np.array([[1, 0, 0, 0]], np.float32), periodic=3)
    g.source_set(0, [0.5, 0.5, 0.5])
    g.transport(N, 6)
    st = g.stats_get()
    want = float(scipy.special.expn(2, tau))
    assert abs(st["w_escaped"] / N - want) < 4 * math.sqrt(want * (1 - want) / N)
    with pytest.raises(krp.KrpError) as ei:
        g.sgrid_begin([krp.make_observer(0.3, 0.2, [0.5, 0.5, 0.5], 1.0)])
    assert ei.value.code == krp.ERR_STATE
    # a packet in an empty, fully periodic box stops after 4096 face crossings instead of flying forever
    g2 = krp.Grid(4, 4, 4, [0, 1, 0, 1, 0, 1], np.zeros((4, 4, 4), np.float32), None, mu, np.array([[1, 0, 0, 0]], np.float32), periodic=7)
    g2.source_set(2, [0.3, 0.4, 0.5], direction=[1, 0, 0])
    g2.transport(100, 1)
    st2 = g2.stats_get()
    assert st2["w_escaped"] == 100 and st2["steps_transport"] == 100 * (3 + 4096 * 4)
    g.close(); g2.close()


def test_thermal_image_of_a_periodic_slab():
    from paper_2512_01283_b200 import krp
    tau = float(np.float32(0.8))
    dens = np.full((3, 6, 6), tau, np.float32)
    mu = np.tile(np.array([1.0, 0.0, 0.0, 0.0], np.float32), (5, 1))
    g = krp.Grid(6, 6, 3, [0, 2, 0, 2, 0, 1], dens, None, mu, np.array([[1, 0, 0, 0]], np.float32), periodic=3)
    o = [krp.make_observer(math.radians(50), math.radians(20), [1, 1, 0.5], 3.0)]
    g.image_rays(o, 8, 8, emis=np.full((3, 6, 6), 1.7, np.float32))
    img = g.image_get()
    c = math.cos(math.radians(50))
    want = float(np.float32(1.7)) * (1 - math.exp(-tau / c)) * (6.0 / 8) ** 2
    assert np.allclose(img[0, 0], want, rtol=1e-12) and np.abs(img[0, 1:]).max() < 1e-15 * want
    g.close()
