"""Shared test helpers (no method arithmetic)."""
import numpy as np

import oracle as orc
from paper_2606_29794_b200 import scenes


def ocfg(scene, **kw):
    """oracle Config for a scene dict."""
    return orc.Config(order=scene["order"], n_gauss=scene["n_gauss"], n_views=scene["n_views"], sh_degree=scene["sh_degree"], **kw)


def oracle_mask(cfg, scene):
    """(bits, active_tiles, slot_of_tile) from the scene's analytic mask descriptor, or (None, None, None)."""
    if scene["mask"] is None:
        return None, None, None
    bits = orc.mask_bits(cfg.order, scene["mask"]["kind"], scene["mask"]["params"])
    act, slot = orc.mask_tiles(cfg, bits)
    return bits, act, slot


def canon_pairs(offsets, keys, vals):
    """Pairs before the sort: the pairs of one (view, Gaussian) are contiguous (offsets[i]..offsets[i+1]) and its tiles are
    distinct, but their order inside the segment is the library's choice (include/uts.h, uts_tile_query).  Returns (keys, vals)
    with every segment sorted by key, the form in which two implementations are compared bit for bit."""
    off = np.asarray(offsets).astype(np.int64)
    n = int(off[-1])
    seg = np.repeat(np.arange(off.shape[0] - 1), np.diff(off))
    order = np.lexsort((np.asarray(keys)[:n], seg))
    return np.asarray(keys)[:n][order], np.asarray(vals)[:n][order]


def small_scene(cfg_id, n_gauss, order, seed=0, **kw):
    return scenes.make_scene(cfg_id, seed=seed, n_gauss=n_gauss, order=order, **kw)


def oracle_on_tiles(oc, scene, pick, bits=None):
    """Oracle forward state restricted to the tiles `pick` (sorted tile ids) but with their COMPLETE lists: every Gaussian is
    preprocessed, a conservative angular pre-filter (plain numpy on the oracle's own records) selects the Gaussians that can
    reach a picked tile, and the oracle's own tile query decides.  Returns dict(proj, sact, skeys, svals, ranges, color, alpha,
    n_last, margin)."""
    pr = orc.preprocess(oc, scene["means"], scene["scales"], scene["quats"], scene["opac"], scene["sh"], scene["W"], scene["b"])
    P, V = oc.n_gauss, oc.n_views
    pick = np.asarray(pick, np.int64)
    sact = pick.astype(np.uint32)
    sslot = np.full(oc.n_tiles, -1, np.int32); sslot[pick] = np.arange(pick.shape[0], dtype=np.int32)
    _, _, tc = orc.centers(oc.tile_order, which=2)
    reach = pr.rs.astype(np.float64) + orc.rho_max_closed(oc.tile_order + oc.query_refine_log2) + orc.rho_max_closed(oc.tile_order) + 1e-6
    cand = np.zeros(P, bool)
    for v in range(V):
        d = pr.dir[v].astype(np.float64) @ tc[pick].T
        cand |= (np.arccos(np.clip(d, -1, 1)) <= reach[v][:, None]).any(axis=1)
    cand_ids = np.flatnonzero(cand).astype(np.int32)
    _, keys, vals, info = orc.tile_query(oc, pr, sslot, gauss_subset=cand_ids)
    sk, sv = orc.sort_pairs(keys, vals)
    rg = orc.tile_ranges(oc, sk)
    col, al, nl, margin, ctr = orc.render_fwd(oc, pr, rg, sv, sact, bits)
    return dict(proj=pr, sact=sact, skeys=sk, svals=sv, ranges=rg, color=col, alpha=al, n_last=nl, margin=margin, qinfo=info, counters=ctr)
