"""Shared test plumbing: build the oracle model and the CUDA grid from one config dict
(paper_2512_01283_b200.inputs) and compare their outputs.  No arithmetic of the method here."""
import numpy as np

from oracle import OracleModel, OracleEvents, OracleStats, OracleZTable, Observer as OraObserver


def oracle_model(cfg, variant=None):
    """variant: None = the oracle proper (fp32 state, R12), "pure" = the control build without those roundings."""
    m = OracleModel(cfg["nx"], cfg["ny"], cfg["nz"], cfg["bounds"], cfg["density"], cfg["bfield"], cfg["mueller"],
                    cfg["opacity"], w_min=cfg["w_min"], max_scatter=cfg["max_scatter"], variant=variant)
    s = cfg["source"]
    m.source_set(s["kind"], s["pos"], s["dir"], s.get("cell_weight"), s.get("emit_records", 0))
    if cfg.get("periodic"):
        m.set_periodic(cfg["periodic"])
    if cfg.get("ztable") is not None:
        m.set_ztable(OracleZTable(cfg["ztable"], variant=variant))
    return m


def oracle_observers(cfg):
    return [OraObserver.make(o["theta"], o["phi"], o["center"], o["half_w"], o["half_h"]) for o in cfg["observers"]]


def oracle_run(cfg, id0, n, cap=None, image=True, flags=0, variant=None):
    """Transport ids [id0, id0+n) and image them.  Returns (events dict sorted by (id,k), img, img2, stats)."""
    m = oracle_model(cfg, variant)
    ev = OracleEvents(cap or max(1024, 16 * n))
    st = OracleStats()
    m.transport(id0, n, cfg["seed"], ev, st)
    assert st.overflow == 0
    img = img2 = None
    if image:
        img, img2, _ = m.image(ev, oracle_observers(cfg), cfg["npix"], cfg["npix"], flags=flags, stats=st)
    k = ev.n
    order = np.lexsort((ev.k[:k], ev.id[:k]))
    out = dict(id=ev.id[:k][order], k=ev.k[:k][order], cell=ev.cell[:k][order], pos=ev.p[:k][order],
               dir=ev.n_in[:k][order], stokes=ev.S[:k][order])
    return out, img, img2, st.as_dict()


def gpu_grid(cfg, device="cuda", host_inputs=False):
    import torch
    from paper_2512_01283_b200 import krp
    if host_inputs:
        dens, bf = cfg["density"], cfg["bfield"]
    else:
        dens = torch.from_numpy(cfg["density"]).to(device)
        bf = None if cfg["bfield"] is None else torch.from_numpy(cfg["bfield"]).to(device)
    g = krp.Grid(cfg["nx"], cfg["ny"], cfg["nz"], cfg["bounds"], dens, bf, cfg["mueller"], cfg["opacity"],
                 w_min=cfg["w_min"], max_scatter=cfg["max_scatter"], periodic=cfg.get("periodic", 0))
    s = cfg["source"]
    w = s.get("cell_weight")
    if w is not None:
        w = torch.from_numpy(np.ascontiguousarray(w, np.float32).ravel()).to(device)
    g.source_set(s["kind"], s["pos"], s["dir"], w, s.get("emit_records", 0))
    if cfg.get("ztable") is not None:
        g.zmatrix_set(cfg["ztable"])
    return g


def gpu_observers(cfg):
    from paper_2512_01283_b200 import krp
    return [krp.make_observer(o["theta"], o["phi"], o["center"], o["half_w"], o["half_h"]) for o in cfg["observers"]]


def gpu_events_sorted(g):
    ev = g.events_get()
    order = np.lexsort((ev["k"], ev["id"]))
    return {k: v[order] for k, v in ev.items()}


def compare_sequences(ora, gpu, ids, stokes_tol=1e-4, pos_tol=2e-3):
    """Per-packet comparison (reading R15): a packet agrees when both sides have the same number of events,
    the same cell at every event, and every Stokes vector within stokes_tol of the oracle's (|dS|_2 / I).
    On top of the north_star's criterion the cell-local positions must agree within pos_tol (fraction of a cell)
    and the directions within 1e-5.
    Returns (fraction of packets that agree, dict of diagnostics; info["good"] is the per-packet mask and the
    fail_* entries count the packets lost to each criterion, in the order they are tested)."""
    ids = np.asarray(ids, np.uint64)
    n = len(ids)
    assert n and np.all(np.diff(ids.astype(np.int64)) == 1), "ids must be a contiguous range"
    id0 = int(ids[0])

    def per_packet(ev):
        idx = (ev["id"].astype(np.int64) - id0) if len(ev["id"]) else np.zeros(0, np.int64)
        assert np.all((idx >= 0) & (idx < n)), "events outside the id range"
        return np.bincount(idx, minlength=n).astype(np.int64), idx
    co, io = per_packet(ora)
    cg, ig = per_packet(gpu)
    good = co == cg
    fail = dict(count=int((~good).sum()), cell=0, stokes=0, pos=0, dir=0)
    # events are sorted by (id, k): for packets with equal counts the j-th events line up
    starts_o = np.concatenate([[0], np.cumsum(co)[:-1]])
    starts_g = np.concatenate([[0], np.cumsum(cg)[:-1]])
    order_o = np.argsort(io, kind="stable")
    order_g = np.argsort(ig, kind="stable")
    worst_s = worst_p = 0.0
    n_ev_cmp = 0
    for p in np.nonzero(good)[0]:
        c = co[p]
        if c == 0:
            continue
        eo = order_o[starts_o[p]:starts_o[p] + c]
        eg = order_g[starts_g[p]:starts_g[p] + c]
        if not (np.array_equal(ora["k"][eo], gpu["k"][eg]) and np.array_equal(ora["cell"][eo], gpu["cell"][eg])):
            good[p] = False
            fail["cell"] += 1
            continue
        So, Sg = ora["stokes"][eo], gpu["stokes"][eg].astype(np.float64)
        ds = np.linalg.norm(So - Sg, axis=1) / So[:, 0]
        dp = np.abs(ora["pos"][eo] - gpu["pos"][eg].astype(np.float64)).max()
        dn = np.abs(ora["dir"][eo] - gpu["dir"][eg].astype(np.float64)).max()
        if ds.max() > stokes_tol:
            good[p] = False; fail["stokes"] += 1
        elif dp > pos_tol:
            good[p] = False; fail["pos"] += 1
        elif dn > 1e-5:
            good[p] = False; fail["dir"] += 1
        else:
            worst_s = max(worst_s, float(ds.max()))
            worst_p = max(worst_p, float(dp))
        n_ev_cmp += c
    return float(good.mean()), dict(n_packets=n, agree=int(good.sum()), worst_stokes=worst_s, worst_pos=worst_p,
                                    events_oracle=int(co.sum()), events_gpu=int(cg.sum()), events_compared=int(n_ev_cmp),
                                    fail=fail, bad_ids=[int(ids[i]) for i in np.nonzero(~good)[0][:8]], good=good)


def show(info):
    return {k: v for k, v in info.items() if k != "good"}


# ------------------------------------------------------------------------------------------
# image comparison of the same packet ids (R15)
# ------------------------------------------------------------------------------------------
def pixels_of(cfg, cell, pos, npx, npy):
    """Test-side restatement of the projection R14 (numpy, fp64): pixel index iy*npx+ix, or -1 outside the frame, of
    events at (cell, cell-local pos) for every observer.  Returns [n_obs, n_events]."""
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    b = np.asarray(cfg["bounds"], np.float64)
    lo = b[0::2]; d = (b[1::2] - b[0::2]) / np.array([nx, ny, nz])
    cell = np.asarray(cell, np.int64)
    idx = np.stack([cell % nx, (cell // nx) % ny, cell // (nx * ny)], 1).astype(np.float64)
    x = lo + (idx + np.asarray(pos, np.float64)) * d
    out = np.zeros((len(cfg["observers"]), len(cell)), np.int64)
    for o, ob in enumerate(cfg["observers"]):
        th, ph = ob["theta"], ob["phi"]
        tv = np.array([np.cos(th) * np.cos(ph), np.cos(th) * np.sin(ph), -np.sin(th)])
        pv = np.array([-np.sin(ph), np.cos(ph), 0.0])
        r = x - np.asarray(ob["center"], np.float64)
        ix = np.floor((r @ pv / ob["half_w"] + 1.0) * npx / 2.0).astype(np.int64)
        iy = np.floor((-(r @ tv) / ob["half_h"] + 1.0) * npy / 2.0).astype(np.int64)
        inside = (ix >= 0) & (ix < npx) & (iy >= 0) & (iy < npy)
        out[o] = np.where(inside, iy * npx + ix, -1)
    return out


def oracle_map_of_ids(cfg, ids, npx, npy, flags=0):
    """Oracle image (and second moments) of the listed packet ids alone."""
    m = oracle_model(cfg)
    ev = OracleEvents(max(1024, 80 * len(ids)))
    st = OracleStats()
    for i in ids:
        m.transport(int(i), 1, cfg["seed"], ev, st)
    assert st.overflow == 0
    img, img2, _ = m.image(ev, oracle_observers(cfg), npx, npy, flags=flags, stats=st)
    return img, img2


def gpu_map_of_ids(cfg, ids, npx, npy, flags=0):
    """CUDA image of the listed packet ids alone (one krp_transport call per id: results do not depend on batching)."""
    g = gpu_grid(cfg)
    g.events_reserve(max(1024, 80 * len(ids)))
    for i in ids:
        g.packet_id_set(int(i))
        g.transport(1, cfg["seed"])
    g.image(gpu_observers(cfg), npx, npy, flags=flags)
    img = g.image_get()
    g.close()
    return img


def compare_images_same_ids(cfg, ora, gev, info, ids, img_g, img_o, img2_o, npx, npy, flags=0, name="", rel=1e-4):
    """The maps of the SAME packet ids from both implementations (R15).
      (1) integrated I, Q, U within 0.5 % (north_star);
      (2) deterministic: with the packets that disagree (sequence comparison) or whose contribution lands in another pixel
          (event positions agree only to rounding, so a contribution on a pixel edge can fall either way) taken out of
          BOTH maps -- their own maps are computed by either implementation from those ids alone -- every pixel of every
          Stokes map agrees within rel * I_pixel;
      (3) the plain north_star form, |dS| <= 3 sigma per pixel with sigma from the oracle's second moments, holds in every
          pixel that no such packet touches (it cannot hold where one implementation deposits a contribution the other
          puts elsewhere: sigma is an estimate from the contributions the oracle has in that pixel, zero if it has none).
    Returns a dict of diagnostics."""
    ids = np.asarray(ids, np.uint64)
    good = info["good"].copy()
    id0 = int(ids[0])
    # (a) contributions of agreeing packets that land in different pixels on the two sides
    go = good[(ora["id"].astype(np.int64) - id0)]
    gg = good[(gev["id"].astype(np.int64) - id0)]
    po = pixels_of(cfg, ora["cell"][go], ora["pos"][go], npx, npy)
    pg = pixels_of(cfg, gev["cell"][gg], gev["pos"][gg].astype(np.float64), npx, npy)
    assert po.shape == pg.shape                                   # same events, same order (sorted by id, k)
    cross = (po != pg).any(axis=0)
    cross_ids = np.unique(ora["id"][go][cross])
    bad_ids = np.union1d(ids[~good], cross_ids).astype(np.uint64)
    out = dict(n_disagree=int((~good).sum()), n_edge=int(len(cross_ids)), n_out=int(len(bad_ids)))
    I_o = img_o[:, 0].sum()
    for s, lab in enumerate("IQU"):
        tot_o, tot_g = img_o[:, s].sum(), img_g[:, s].sum()
        assert abs(tot_g - tot_o) <= 0.005 * max(abs(tot_o), 1e-3 * I_o), (name, lab, tot_g, tot_o)
    if len(bad_ids):
        G_bad = gpu_map_of_ids(cfg, bad_ids, npx, npy, flags)
        O_bad, _ = oracle_map_of_ids(cfg, bad_ids, npx, npy, flags)
    else:
        G_bad = np.zeros_like(img_g); O_bad = np.zeros_like(img_o)
    A, B = img_g - G_bad, img_o - O_bad
    floor = 1e-9 * img_o[:, 0].max()
    tol = rel * np.abs(B[:, :1]) + floor
    err = np.abs(A - B)
    worst = float((err / (np.abs(B[:, :1]) + floor / rel)).max())
    out["worst_rel"] = worst
    n_bad = int((err > tol).sum())
    assert n_bad == 0, (name, "deterministic same-id check", n_bad, worst, out)
    touched = ((G_bad != 0) | (O_bad != 0)).any(axis=1, keepdims=True)
    sigma = np.sqrt(img2_o)
    fail3 = np.abs(img_g - img_o) > 3 * sigma + floor
    out["pixels_3sigma_fail_touched"] = int((fail3 & touched).sum())
    assert int((fail3 & ~touched).sum()) == 0, (name, "3 sigma per pixel outside touched pixels", int((fail3 & ~touched).sum()))
    out["pixels_touched"] = int(touched.sum())
    return out
