"""Shared test plumbing: build the oracle model and the CUDA grid from one config dict
(paper_2512_01283_b200.inputs) and compare their outputs.  No arithmetic of the method here."""
import numpy as np

from oracle import OracleModel, OracleEvents, OracleStats, Observer as OraObserver


def oracle_model(cfg):
    m = OracleModel(cfg["nx"], cfg["ny"], cfg["nz"], cfg["bounds"], cfg["density"], cfg["bfield"], cfg["mueller"],
                    cfg["opacity"], w_min=cfg["w_min"], max_scatter=cfg["max_scatter"])
    s = cfg["source"]
    m.source_set(s["kind"], s["pos"], s["dir"], s.get("cell_weight"), s.get("emit_records", 0))
    return m


def oracle_observers(cfg):
    return [OraObserver.make(o["theta"], o["phi"], o["center"], o["half_w"], o["half_h"]) for o in cfg["observers"]]


def oracle_run(cfg, id0, n, cap=None, image=True, flags=0):
    """Transport ids [id0, id0+n) and image them.  Returns (events dict sorted by (id,k), img, img2, stats)."""
    m = oracle_model(cfg)
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
                 w_min=cfg["w_min"], max_scatter=cfg["max_scatter"])
    s = cfg["source"]
    w = s.get("cell_weight")
    if w is not None:
        w = torch.from_numpy(np.ascontiguousarray(w, np.float32).ravel()).to(device)
    g.source_set(s["kind"], s["pos"], s["dir"], w, s.get("emit_records", 0))
    return g


def gpu_observers(cfg):
    from paper_2512_01283_b200 import krp
    return [krp.make_observer(o["theta"], o["phi"], o["center"], o["half_w"], o["half_h"]) for o in cfg["observers"]]


def gpu_events_sorted(g):
    ev = g.events_get()
    order = np.lexsort((ev["k"], ev["id"]))
    return {k: v[order] for k, v in ev.items()}


def compare_sequences(ora, gpu, ids, stokes_tol=1e-4, pos_tol=1e-2):
    """Per-packet comparison (reading R15): a packet agrees when both sides have the same number of events,
    the same cell at every event, and every Stokes vector within stokes_tol of the oracle's (|dS|_2 / I).
    On top of the north_star's criterion the cell-local positions must agree within pos_tol (fraction of a cell)
    and the directions within 1e-5.
    Returns (fraction of packets that agree, dict of diagnostics)."""
    ids = np.asarray(ids, np.uint64)
    n = len(ids)
    rank = {int(v): i for i, v in enumerate(ids)}

    def per_packet(ev):
        cnt = np.zeros(n, np.int64)
        idx = np.array([rank[int(v)] for v in ev["id"]], np.int64) if len(ev["id"]) else np.zeros(0, np.int64)
        np.add.at(cnt, idx, 1)
        return cnt, idx
    co, io = per_packet(ora)
    cg, ig = per_packet(gpu)
    good = co == cg
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
            continue
        So, Sg = ora["stokes"][eo], gpu["stokes"][eg].astype(np.float64)
        ds = np.linalg.norm(So - Sg, axis=1) / So[:, 0]
        dp = np.abs(ora["pos"][eo] - gpu["pos"][eg].astype(np.float64)).max()
        dn = np.abs(ora["dir"][eo] - gpu["dir"][eg].astype(np.float64)).max()
        if ds.max() > stokes_tol or dp > pos_tol or dn > 1e-5:
            good[p] = False
        worst_s = max(worst_s, float(ds.max()))
        worst_p = max(worst_p, float(dp))
        n_ev_cmp += c
    return float(good.mean()), dict(n_packets=n, agree=int(good.sum()), worst_stokes=worst_s, worst_pos=worst_p,
                                    events_oracle=int(co.sum()), events_gpu=int(cg.sum()), events_compared=int(n_ev_cmp),
                                    bad_ids=[int(ids[i]) for i in np.nonzero(~good)[0][:8]])
