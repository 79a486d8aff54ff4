"""GPU parity of the full aligned-grain scattering matrix path (reading R21):
rejection sampling against Z and the Z peel-off on the GPU against the oracle, event by event and map by map."""
import numpy as np
import pytest

from paper_2512_01283_b200 import inputs, krp
from harness import (oracle_run, gpu_grid, gpu_observers, gpu_events_sorted, compare_sequences, compare_images_same_ids, show)

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name,apar,aperp", [("c4", 0.6 + 0.2j, 1.0 + 0.05j), ("c5", 1.0, 1.0), ("c3", 0.3, 1.0)])
def test_zmatrix_sequences_and_images(name, apar, aperp):
    kw = dict(c4=dict(n=20, n_packets=5000, npix=32), c5=dict(n=16, n_packets=3000, npix=24), c3=dict(n=8, n_packets=1200, npix=16))[name]
    cfg = inputs.make(name, **kw)
    cfg["ztable"] = inputs.dipole_ztable(37, 37, 72, a_par=apar, a_perp=aperp)
    n = cfg["n_packets"]
    ora, img_o, img2_o, st_o = oracle_run(cfg, 0, n, cap=64 * n)
    g = gpu_grid(cfg)
    g.events_reserve(64 * n)
    g.transport(n, cfg["seed"])
    gev = gpu_events_sorted(g)
    frac, info = compare_sequences(ora, gev, np.arange(n))
    print("zmatrix", name, frac, show(info))
    assert frac >= 0.999, show(info)
    g.image(gpu_observers(cfg), cfg["npix"], cfg["npix"])
    img_g = g.image_get()
    compare_images_same_ids(cfg, ora, gev, info, np.arange(n), img_g, img_o, img2_o, cfg["npix"], cfg["npix"], name="zmatrix-" + name)
    st = g.stats_get()
    assert abs(st["w_escaped"] + st["w_absorbed"] + st["w_cut"] - st["w_emitted"]) <= 1e-5 * n
    # back to F(Theta): a different problem (except for isotropic dipoles, which ARE Rayleigh scattering -- but the table then differs)
    g.zmatrix_set(None)
    g.stats_reset(); g.packet_id_set(0)
    g.transport(n, cfg["seed"])
    ev2 = gpu_events_sorted(g)
    assert len(ev2["id"]) != len(gev["id"]) or not np.array_equal(ev2["cell"], gev["cell"])
    g.close()


def test_zmatrix_argument_errors():
    cfg = inputs.make("c1", n=8, n_packets=10, npix=8)
    g = gpu_grid(cfg)                                       # 4-byte cells: no field to define a grain frame
    with pytest.raises(krp.KrpError) as ei:
        g.zmatrix_set(inputs.dipole_ztable(5, 5, 8))
    assert ei.value.code == krp.ERR_ARG
    cfg = inputs.make("c4", n=8, n_packets=10, npix=8)
    g = gpu_grid(cfg)
    bad = inputs.dipole_ztable(5, 5, 8); bad[1, 2, 3, 0, 0] = -1.0
    with pytest.raises(krp.KrpError):
        g.zmatrix_set(bad)
    g.zmatrix_set(inputs.dipole_ztable(5, 5, 8))
    with pytest.raises(krp.KrpError) as ei:
        g.sgrid_begin(gpu_observers(cfg))
    assert ei.value.code == krp.ERR_STATE
    g.close()
