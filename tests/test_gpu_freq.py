"""GPU parity of the frequency-bin axis (eq. 8 holds per frequency bin).  Bins are
independent problems on the same dust: bin b has its own tables and kappa*rho = kappa_scale[b] x the model's.  The oracle
of bin b is therefore the pinned oracle run on (density x kappa_scale[b] in fp32, tables of b); the CUDA path must match it
event by event and map by map for every bin, with the bins' maps kept apart."""
import numpy as np
import pytest

from paper_2512_01283_b200 import inputs, krp
from harness import (oracle_run, gpu_grid, gpu_observers, gpu_events_sorted, compare_sequences, compare_images_same_ids, show)

pytestmark = pytest.mark.gpu


def _bins(general):
    if general:
        return [(inputs.hg_mueller(0.3, 0.4, seed=11), inputs.aligned_opacity(1.1, 0.02, 0.5), 0.6),
                (inputs.hg_mueller(0.6, 0.25, seed=12), inputs.aligned_opacity(1.3, -0.05, 0.8), 1.0),
                (inputs.rayleigh_mueller(), inputs.aligned_opacity(1.02, 0.0, 0.3), 2.5)]
    return [(inputs.rayleigh_mueller(), inputs.constant_opacity(1.0, 0.5), 1.0),
            (inputs.hg_mueller(0.5, 0.4, seed=13), inputs.constant_opacity(0.7, 0.9), 3.0)]


@pytest.mark.parametrize("name", ["c4", "c1"])
def test_every_bin_matches_its_oracle(name):
    general = name == "c4"
    cfg = inputs.make(name, n=20, n_packets=5000, npix=32)
    bins = _bins(general)
    n = cfg["n_packets"]
    g = gpu_grid(cfg)
    g.freq_define([(mu, op, cfg["w_min"], cfg["max_scatter"]) for mu, op, k in bins], [k for _, _, k in bins])
    obs = gpu_observers(cfg)
    maps = []
    for b in (1, 0, 2)[:len(bins)] if general else (1, 0):
        mu, op, k = bins[b]
        cfg_b = dict(cfg, mueller=mu, opacity=op, density=(cfg["density"] * np.float32(k)).astype(np.float32))
        ora, img_o, img2_o, st_o = oracle_run(cfg_b, 0, n, cap=64 * n)
        g.freq_select(b)
        g.packet_id_set(0)
        g.events_reserve(64 * n)
        g.transport(n, cfg["seed"])
        gev = gpu_events_sorted(g)
        frac, info = compare_sequences(ora, gev, np.arange(n))
        print(name, "bin", b, frac, show(info))
        assert frac >= 0.999, show(info)
        g.image(obs, cfg["npix"], cfg["npix"])
        img_g = g.image_get()
        compare_images_same_ids(cfg_b, ora, gev, info, np.arange(n), img_g, img_o, img2_o, cfg["npix"], cfg["npix"], name="bin%d" % b)
        maps.append((b, img_g.copy()))
    # the bins' maps are kept apart: coming back to a bin finds its map untouched
    for b, img in maps:
        g.freq_select(b)
        assert np.array_equal(g.image_get(), img)
    assert not np.allclose(maps[0][1], maps[1][1])
    # errors: a bin cannot be left with events in the buffer; a bad bin index; a dichroic table on a 4-byte-cell model
    g.freq_select(0)
    g.transport(100, 1)
    with pytest.raises(krp.KrpError) as ei:
        g.freq_select(1)
    assert ei.value.code == krp.ERR_STATE
    g.events_clear()
    with pytest.raises(krp.KrpError):
        g.freq_select(len(bins))
    if not general:
        with pytest.raises(krp.KrpError) as ei:
            g.freq_define([(inputs.rayleigh_mueller(), inputs.aligned_opacity(), 1e-4, 64)], [1.0])
        assert ei.value.code == krp.ERR_ARG
    g.close()


def test_grid_update_keeps_the_bins():
    """A new density snapshot (krp_grid_update) under frequency bins: the current bin's factor is applied to the new values."""
    cfg = inputs.make("c4", n=16, n_packets=3000, npix=24)
    bins = _bins(True)[:2]
    g = gpu_grid(cfg)
    g.freq_define([(mu, op, cfg["w_min"], cfg["max_scatter"]) for mu, op, k in bins], [k for _, _, k in bins])
    g.freq_select(1); g.freq_select(0)
    dens2 = (cfg["density"] * 1.7).astype(np.float32)
    g.update(dens2, cfg["bfield"])
    g.transport(cfg["n_packets"], cfg["seed"])
    ev = gpu_events_sorted(g)
    mu, op, k = bins[0]
    cfg_b = dict(cfg, mueller=mu, opacity=op, density=(dens2 * np.float32(k)).astype(np.float32))
    ora, _, _, _ = oracle_run(cfg_b, 0, cfg["n_packets"], cap=64 * cfg["n_packets"], image=False)
    frac, info = compare_sequences(ora, ev, np.arange(cfg["n_packets"]))
    assert frac >= 0.999, show(info)
    g.close()


def test_bins_and_an_open_source_grid_do_not_mix():
    """A source grid holds the deposits of the bin it was opened in: selecting another bin while it is open is refused."""
    cfg = inputs.make("c1", n=12, n_packets=500, npix=16)
    bins = _bins(False)
    g = gpu_grid(cfg)
    g.freq_define([(mu, op, cfg["w_min"], cfg["max_scatter"]) for mu, op, k in bins], [k for _, _, k in bins])
    g.sgrid_begin(gpu_observers(cfg))
    with pytest.raises(krp.KrpError) as ei:
        g.freq_select(1)
    assert ei.value.code == krp.ERR_STATE and "source grid" in str(ei.value)
    g.freq_select(0)                      # the current bin: nothing to do
    g.sgrid_end()
    g.freq_select(1)
    g.close()
