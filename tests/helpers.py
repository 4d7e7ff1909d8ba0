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


def small_scene(cfg_id, n_gauss, order, seed=0, **kw):
    return scenes.make_scene(cfg_id, seed=seed, n_gauss=n_gauss, order=order, **kw)
