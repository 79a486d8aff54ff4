"""krp_image_events_noalloc (include/krp.h): the imaging entry point that allocates nothing -- its event records and
control block live in one fixed device array inside the library -- against the existing path, krp_image, on the same
events.  Collected last (file name): the suite runs with pytest -x.

Tolerance: that of test_scheduling_switches_do_not_change_results (tests/test_gpu_parity.py) for maps that are "equal to
the rounding of the fp32 march": per pixel and Stokes component 2e-5 x the brightest pixel, 1e-6 on the summed I.  (The
public event format carries W(1,q,u,v) in fp32, from which the entry point re-derives q,u,v, and general mode marches
over the 16-byte cells instead of krp_image's per-observer coefficient arrays.)
"""
import numpy as np
import pytest

from paper_2512_01283_b200 import inputs
from harness import gpu_grid, gpu_observers

pytestmark = pytest.mark.gpu

CASES = {
    "c2": dict(n=32, n_packets=20000, npix=32),        # scalar cells, point source, HG table with S34
    "c4": dict(n=24, n_packets=6000, npix=32),         # general cells, helical field, volume source, 3 observers
}


def _close(img, ref):
    scale = np.abs(ref[0]).max()
    for s in range(4):
        assert np.abs(img[s] - ref[s]).max() <= 2e-5 * scale, s
    assert abs(img[0].sum() - ref[0].sum()) <= 1e-6 * ref[0].sum()


@pytest.mark.parametrize("name", sorted(CASES))
def test_no_alloc_imaging_equals_krp_image(name):
    import torch
    from paper_2512_01283_b200 import krp
    cfg = inputs.make(name, **CASES[name])
    npix = cfg["npix"]
    g = gpu_grid(cfg)
    g.transport(cfg["n_packets"], cfg["seed"])
    ev = g.events_get()                      # before krp_image, which consumes the buffer
    n = len(ev["k"])
    assert 1000 < n <= krp.NOALLOC_MAX_EVENTS
    obs = gpu_observers(cfg)
    assert len(obs) >= 2
    g.image(obs, npix, npix)
    ref = g.image_get()                      # the existing path: [n_obs][4][npy][npx]
    assert ref[:, 0].sum() > 0

    dev = "cuda"
    k = torch.from_numpy(ev["k"].astype(np.int32)).to(dev)
    cell = torch.from_numpy(ev["cell"].astype(np.int64)).to(dev)
    pos = torch.from_numpy(np.ascontiguousarray(ev["pos"], np.float32)).to(dev)
    dr = torch.from_numpy(np.ascontiguousarray(ev["dir"], np.float32)).to(dev)
    st = torch.from_numpy(np.ascontiguousarray(ev["stokes"], np.float32)).to(dev)
    imgs = [torch.zeros(4, npix, npix, dtype=torch.float64, device=dev) for _ in range(4)]
    torch.cuda.synchronize()

    # two calls in a row, all events, two different observers: the second must not see anything of the first
    g.image_events_noalloc(k, cell, pos, dr, st, obs[0], npix, npix, imgs[0])
    g.image_events_noalloc(k, cell, pos, dr, st, obs[1], npix, npix, imgs[1])
    torch.cuda.synchronize()
    _close(imgs[0].cpu().numpy(), ref[0])
    _close(imgs[1].cpu().numpy(), ref[1])

    # the same observer again in two parts of unequal size added into one map (a call with fewer events than the one
    # before it: the records the earlier call left beyond n are not read), device memory unchanged over the calls
    free0 = torch.cuda.mem_get_info()[0]
    h = n // 3
    g.image_events_noalloc(k[:h], cell[:h], pos[:h], dr[:h], st[:h], obs[0], npix, npix, imgs[2])
    g.image_events_noalloc(k[h:], cell[h:], pos[h:], dr[h:], st[h:], obs[0], npix, npix, imgs[2])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    _close(imgs[2].cpu().numpy(), ref[0])

    # events the entry point must leave out are counted and contribute nothing
    cell_bad = cell.clone()
    cell_bad[5] = -1
    cell_bad[7] = cfg["nx"] * cfg["ny"] * cfg["nz"]
    st_bad = st.clone()
    st_bad[5] = 1e30
    st_bad[7] = 1e30
    rej = g.image_events_noalloc(k, cell_bad, pos, dr, st_bad, obs[0], npix, npix, imgs[3], want_rejected=True)
    assert rej == 2
    keep = np.ones(n, bool)
    keep[[5, 7]] = False
    ks, cs, ps, ds, ss = (torch.from_numpy(np.ascontiguousarray(a[keep])).to(dev) for a in
                          (ev["k"].astype(np.int32), ev["cell"].astype(np.int64), ev["pos"].astype(np.float32),
                           ev["dir"].astype(np.float32), ev["stokes"].astype(np.float32)))
    img_keep = torch.zeros(4, npix, npix, dtype=torch.float64, device=dev)
    assert g.image_events_noalloc(ks, cs, ps, ds, ss, obs[0], npix, npix, img_keep, want_rejected=True) == 0
    a, b = imgs[3].cpu().numpy(), img_keep.cpu().numpy()
    assert np.allclose(a, b, rtol=1e-11, atol=1e-13 * b[0].max())

    # the grid's own state is untouched: a second pass of the existing path gives the first one's maps again
    g.image_reset()
    g.packet_id_set(0)
    g.transport(cfg["n_packets"], cfg["seed"])
    g.image(obs, npix, npix)
    again = g.image_get()
    assert np.allclose(again, ref, rtol=1e-11, atol=1e-13 * ref[:, 0].max())
    g.close()


def test_no_alloc_limits_and_arguments():
    import torch
    from paper_2512_01283_b200 import krp
    cfg = inputs.make("c1", n=8, n_packets=100, npix=8)
    g = gpu_grid(cfg)
    obs = gpu_observers(cfg)[0]
    dev = "cuda"
    n = krp.NOALLOC_MAX_EVENTS + 1
    k = torch.ones(n, dtype=torch.int32, device=dev)
    cell = torch.zeros(n, dtype=torch.int64, device=dev)
    v3 = torch.zeros(n, 3, dtype=torch.float32, device=dev)
    dz = v3.clone()
    dz[:, 2] = 1.0
    v4 = torch.zeros(n, 4, dtype=torch.float32, device=dev)
    img = torch.zeros(4, 8, 8, dtype=torch.float64, device=dev)
    with pytest.raises(krp.KrpError) as e:
        g.image_events_noalloc(k, cell, v3, dz, v4, obs, 8, 8, img)
    assert e.value.code == krp.ERR_ARG and str(krp.NOALLOC_MAX_EVENTS) in str(e.value)
    # the maximum itself is accepted; events of weight 0 leave the map at zero; no events is a no-op
    assert g.image_events_noalloc(k[:-1], cell[:-1], v3[:-1], dz[:-1], v4[:-1], obs, 8, 8, img, want_rejected=True) == 0
    g.image_events_noalloc(k[:0], cell[:0], v3[:0], dz[:0], v4[:0], obs, 8, 8, img)
    # a direction that is no unit vector is left out
    assert g.image_events_noalloc(k[:10], cell[:10], v3[:10], v3[:10], v4[:10], obs, 8, 8, img, want_rejected=True) == 10
    torch.cuda.synchronize()
    assert float(img.abs().max()) == 0.0
    g.close()
