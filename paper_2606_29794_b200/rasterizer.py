"""Buffer management around the seven ABI calls: allocates the caller-owned buffers with torch and runs the stages in
Alg.1's order and the backward.  No arithmetic of the method lives here."""
from __future__ import annotations

import torch

from . import binding as B


def _i64(n, dev): return torch.empty(n, dtype=torch.int64, device=dev)
def _i32(n, dev): return torch.empty(n, dtype=torch.int32, device=dev)
def _f32(*s, dev): return torch.empty(*s, dtype=torch.float32, device=dev)
def _bytes(n, dev): return torch.empty((n + 255) // 256 * 32, dtype=torch.int64, device=dev)   # 256-byte granular, 256-aligned by the allocator


class Rasterizer:
    """Holds every buffer of one configuration.  forward() / backward() enqueue on torch's current stream; the only host
    synchronisation is the pair count returned by uts_tile_query."""

    def __init__(self, cfg: B.Config, mask: B.Mask | None = None, device="cuda", pair_capacity: int = 0, depth_presort: bool = True,
                 fused_lists: bool = True, marks: bool = True, tuning: B.Tuning | None = None):
        B.lib()
        if not torch.cuda.is_available():
            raise RuntimeError("uts: a CUDA device is required (no CPU fallback)")
        self.cfg, self.mask, self.dev = cfg, (mask or B.Mask.full()), device
        self.tuning = tuning                # uts_tuning for the tile query (tests, A/B runs); None = the library's defaults
        V, P = cfg.n_views, cfg.n_gauss
        self.S = self.mask.n_slots(cfg)
        npx = self.S * cfg.ppt
        self.proj = B.Proj.empty(cfg, device)
        self.offsets = _i64(V * P + 1, device)
        # fused_lists: uts_tile_lists (query + sort + ranges in one call, large discs emitted tile-major) instead of the three calls
        self.fused_lists = bool(fused_lists) and depth_presort
        self.tq_scratch = _bytes(B.uts_tile_lists_scratch_bytes(cfg) if self.fused_lists else B.uts_tile_query_scratch_bytes(cfg), device)
        # depth_presort: order the Gaussians by radial depth first so that the pair sort only runs its (view,tile) passes
        self.depth_presort = depth_presort
        self.emit_rank = _i32(max(V * P, 1), device) if depth_presort else None
        self.do_scratch = _bytes(B.uts_depth_order_scratch_bytes(cfg), device) if depth_presort else None
        self.ranges = _i64(V * cfg.n_tiles * 2, device).view(V * cfg.n_tiles, 2)
        self.color = _f32(V, npx, 3, dev=device); self.alpha = _f32(V, npx, dev=device)
        self.trans = _f32(V, npx, dev=device); self.n_last = _i32(V * npx, device).view(V, npx)
        # marks: the forward blend records which (warp, entry) pairs blended anything, the backward visits only those
        self.use_marks = bool(marks)
        self.marks = None
        self.capacity = 0
        self.n_pairs = 0
        self._alloc_pairs(max(int(pair_capacity), 1024))
        self.grads = None

    def _alloc_pairs(self, cap):
        self.keys = self.vals = self.keys_tmp = self.vals_tmp = self.sort_scratch = None
        self.capacity = int(cap)
        d = self.dev
        self.keys, self.keys_tmp = _i64(cap, d), _i64(cap, d)
        self.vals, self.vals_tmp = _i32(cap, d), _i32(cap, d)
        self.sort_scratch = _bytes(B.uts_sort_scratch_bytes(cap), d)
        self.marks = torch.zeros(B.uts_render_marks_bytes(self.cfg, cap) // 4, dtype=torch.int32, device=d) if self.use_marks else None

    # ---- stages (each is one ABI call) -------------------------------------------------------------
    def preprocess(self, g, views): B.uts_preprocess(self.cfg, g, views, self.proj)

    def depth_order(self):
        if self.depth_presort:
            B.uts_depth_order(self.cfg, self.proj.rho, self.emit_rank, self.do_scratch)

    def tile_query(self):
        try:
            self.n_pairs = B.uts_tile_query(self.cfg, self.proj, self.mask, self.offsets, self.keys, self.vals, self.capacity, self.tq_scratch,
                                            self.emit_rank, self.tuning)
        except B.UtsError as e:
            if e.status != B.UTS_ERR_CAPACITY:
                raise
            self._alloc_pairs(int(e.needed * 1.05) + 1024)
            self.n_pairs = B.uts_tile_query(self.cfg, self.proj, self.mask, self.offsets, self.keys, self.vals, self.capacity, self.tq_scratch,
                                            self.emit_rank, self.tuning)
        return self.n_pairs

    def tile_lists(self):
        """uts_tile_lists: sorted keys / vals and ranges in one call (needs the depth order)."""
        args = lambda: (self.cfg, self.proj, self.mask, self.emit_rank, self.keys, self.vals, self.keys_tmp, self.vals_tmp, self.capacity, self.ranges,
                        self.tq_scratch, self.sort_scratch, self.tuning)
        try:
            self.n_pairs = B.uts_tile_lists(*args())
        except B.UtsError as e:
            if e.status != B.UTS_ERR_CAPACITY:
                raise
            self._alloc_pairs(int(e.needed * 1.05) + 1024)
            self.n_pairs = B.uts_tile_lists(*args())
        return self.n_pairs

    def sort(self):
        B.uts_sort(self.cfg, self.n_pairs, self.keys, self.vals, self.keys_tmp, self.vals_tmp, self.sort_scratch, self.depth_presort)
    def tile_ranges(self): B.uts_tile_ranges(self.cfg, self.n_pairs, self.keys, self.ranges)

    def render_fwd(self):
        if self.use_marks:
            B.uts_render_fwd_marked(self.cfg, self.proj, self.mask, self.ranges, self.vals, self.capacity, self.color, self.alpha, self.trans,
                                    self.n_last, self.marks)
        else:
            B.uts_render_fwd(self.cfg, self.proj, self.mask, self.ranges, self.vals, self.color, self.alpha, self.trans, self.n_last)

    def render_fwd_depth(self):
        """Colour + inverse radial depth in one blend pass; returns the depth image [V, S*256]."""
        if getattr(self, "depth", None) is None:
            self.depth = torch.empty_like(self.alpha)
        B.uts_render_fwd_depth(self.cfg, self.proj, self.mask, self.ranges, self.vals, self.capacity, self.color, self.alpha, self.trans, self.n_last,
                               self.depth, self.marks if self.use_marks else None)
        return self.depth

    def render_bwd_depth(self, dL_dcolor, dL_ddepth, dL_dalpha=None):
        """Backward of render_fwd_depth: grads["rgb" / "conic" / "mu2" / "opac"] hold both losses' terms, grads["invr"] = dL/d(1/rho) [V,P]."""
        G = self._alloc_grads()
        if "invr" not in G:
            G["invr"] = _f32(self.cfg.n_views, self.cfg.n_gauss, dev=self.dev)
        B.uts_render_bwd_depth(self.cfg, self.proj, self.mask, self.ranges, self.vals, self.capacity, self.trans, self.n_last,
                               self.marks if self.use_marks else None, dL_dcolor, dL_dalpha, dL_ddepth, G["rgb"], G["conic"], G["mu2"], G["opac"], G["invr"])

    def _alloc_grads(self):
        if self.grads is None:
            V, P, M, d = self.cfg.n_views, self.cfg.n_gauss, self.cfg.n_sh, self.dev
            self.grads = dict(rgb=_f32(V, P, 3, dev=d), conic=_f32(V, P, 3, dev=d), mu2=_f32(V, P, 2, dev=d), opac=_f32(P, dev=d),
                              means=_f32(P, 3, dev=d), scales=_f32(P, 3, dev=d), quats=_f32(P, 4, dev=d), sh=_f32(P, M, 3, dev=d))
        return self.grads

    def render_bwd(self, dL_dcolor, dL_dalpha=None):
        G = self._alloc_grads()
        if self.use_marks:
            B.uts_render_bwd_marked(self.cfg, self.proj, self.mask, self.ranges, self.vals, self.capacity, self.trans, self.n_last, self.marks,
                                    dL_dcolor, dL_dalpha, G["rgb"], G["conic"], G["mu2"], G["opac"])
        else:
            B.uts_render_bwd(self.cfg, self.proj, self.mask, self.ranges, self.vals, self.trans, self.n_last, dL_dcolor, dL_dalpha,
                             G["rgb"], G["conic"], G["mu2"], G["opac"])

    def preprocess_bwd(self, g, views):
        G = self._alloc_grads()
        B.uts_preprocess_bwd(self.cfg, g, views, self.proj.flags, G["rgb"], G["conic"], G["mu2"], G["means"], G["scales"], G["quats"], G["sh"])

    # ---- whole path --------------------------------------------------------------------------------
    def forward(self, g, views):
        self.preprocess(g, views)
        self.depth_order()
        if self.fused_lists:
            self.tile_lists()
        else:
            self.tile_query()
            self.sort()
            self.tile_ranges()
        self.render_fwd()
        return self.color, self.alpha

    def forward_depth_prefix(self, g, views, keep: int):
        """Forward with tile lists built from the `keep` nearest Gaussians of each view only (needs fused_lists).  Returns
        (color, alpha, n_open): n_open = visible pixels that did not saturate; 0 means image, n_last and the gradients of backward()
        are exactly those of the full lists (include/uts.h, uts_depth_prefix_flags).  The caller decides what to do otherwise
        (forward() again, or a larger prefix)."""
        assert self.fused_lists
        self.preprocess(g, views)
        self.depth_order()
        if getattr(self, "_pflags", None) is None:
            self._pflags = torch.empty_like(self.proj.flags)
            self._cnt = torch.zeros(1, dtype=torch.int64, device=self.dev)
        B.uts_depth_prefix_flags(self.cfg, self.proj.flags, self.emit_rank, int(keep), self._pflags)
        full = self.proj
        self.proj = B.Proj(full.dir, full.lonlat, full.rho, full.conic_opac, full.rs, full.rgb, self._pflags)
        try:
            self.tile_lists()
        finally:
            self.proj = full
        self.render_fwd()
        n_open = B.uts_count_unsaturated(self.cfg, self.mask, self.trans, self._cnt)
        return self.color, self.alpha, n_open

    def forward_auto(self, g, views):
        """forward() through the depth prefix when that is known to pay, through the full lists otherwise; the result is always the
        full lists' one (a prefix is accepted only when uts_count_unsaturated returns 0).  The prefix length is a running guess:
        it starts at P/128, grows fourfold after a failed attempt (the full lists are then built for this call) and the attempts stop
        once it would pass P/2 — the scene does not saturate, as configs 1, 2, 3 and 5 do not."""
        P = self.cfg.n_gauss
        st = self.__dict__.setdefault("_auto", dict(keep=max(P // 128, 1), off=not self.fused_lists, used_prefix=False))
        st["used_prefix"] = False
        if not st["off"]:
            c, a, n_open = self.forward_depth_prefix(g, views, st["keep"])
            if n_open == 0:
                st["used_prefix"] = True
                return c, a
            st["keep"] *= 4
            if st["keep"] > P // 2:
                st["off"] = True
        return self.forward(g, views)

    def backward(self, g, views, dL_dcolor, dL_dalpha=None):
        self.render_bwd(dL_dcolor, dL_dalpha)
        self.preprocess_bwd(g, views)
        return self.grads


def scene_to_device(scene, device="cuda"):
    """numpy scene dict (scenes.make_scene) -> (Gaussians, Views) on the device."""
    t = lambda a: torch.from_numpy(a).to(device).contiguous()
    return (B.Gaussians(t(scene["means"]), t(scene["scales"]), t(scene["quats"]), t(scene["opac"]), t(scene["sh"])),
            B.Views(t(scene["W"]), t(scene["b"])))


def config_of(scene, **kw) -> B.Config:
    return B.Config(order=scene["order"], n_gauss=scene["n_gauss"], n_views=scene["n_views"], sh_degree=scene["sh_degree"], **kw)
