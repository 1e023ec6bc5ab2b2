"""Buffer plumbing around the five C-ABI calls: allocation (PyTorch), call order, capacity regrowth.

No arithmetic of the method lives here -- each stage is one call into libxpr.so (binding.py).
Call stack of one step:
    xpr_project -> xpr_bin_sort -> xpr_rasterize_fwd -> [loss outside] -> xpr_rasterize_bwd -> xpr_project_bwd
With cfg["ray_eval"] = 1 (XPR-3DGUT evaluation):
    xpr_pixel_info, xpr_project -> xpr_project_ray -> xpr_bin_sort -> xpr_rasterize_ray_fwd -> [loss] ->
    xpr_rasterize_ray_bwd -> xpr_project_bwd (zero footprint gradients) -> xpr_ray_bwd
"""
from __future__ import annotations

import torch

from . import binding as xb


class SplatPipeline:
    """Owns the intermediate device buffers for one (N, camera, config) and sequences the stages."""

    def __init__(self, N: int, cam, cfg: dict, pair_capacity: int | None = None, device="cuda:0"):
        self.N = int(N)
        self.device = torch.device(device)
        # a list of cameras = a batch of views rendered by ONE call per stage (xpr_config.views; Table 2)
        self.V = len(cam) if isinstance(cam, (list, tuple)) else 1
        if self.V > 1:
            self.cam = xb.make_cameras(cam)
            cam0 = self.cam[0]
            cfg = dict(cfg, views=self.V)
        else:
            cam = cam[0] if isinstance(cam, (list, tuple)) else cam
            self.cam = cam if isinstance(cam, xb.XprCamera) else xb.make_camera(cam)
            cam0 = self.cam
        self.ray_eval = bool(cfg.get("ray_eval", 0)) if isinstance(cfg, dict) else False
        # f3: the compositing pass also renders the depth image and the accumulated opacity (2D evaluation only)
        self.features = bool(cfg.get("features", 0)) if isinstance(cfg, dict) else False
        if self.V > 1 and self.ray_eval:
            raise ValueError("xpr: a batch of views is built for the 2D evaluation (colour, depth and accumulated opacity)")
        self._dL = None
        # overlap_fill: the zero-fill of the parameter gradients (xpr_project_bwd_fill: 236 B per Gaussian of HBM stores without
        # inputs) runs on a second stream, forked at the forward compositing kernel (4, the default), at the compositing
        # backward (1) or at the binning stage (2); 0: inside xpr_project_bwd.  Measured: under the forward
        # kernel -- ALU-bound, no atomics -- the step gets 16 us shorter on configs 3 and 5; under the backward or the
        # binning kernels the host kernel slows down by what the fill saves.
        self.overlap_fill = int(cfg.get("overlap_fill", 4)) if isinstance(cfg, dict) else 4
        self._filled = False
        # fuse_loss: step_async() forms dL/dimage of the two configured losses inside the compositing backward
        # (xpr_rasterize_bwd_loss) instead of a separate xpr_loss_grad pass; colour pass of the 2D evaluation only
        self.fuse_loss = bool(cfg.get("fuse_loss", 1)) if isinstance(cfg, dict) else True
        # f3: constant (dL/dD, dL/dA) of a loss that is linear in the features; step_async() feeds them to the backward
        self.feature_grads = None
        self.cfg = cfg if isinstance(cfg, xb.XprConfig) else xb.make_config(cfg)
        self.K = (int(self.cfg.sh_degree) + 1) ** 2
        self.W, self.H = int(cam0.width), int(cam0.height)
        self.TW, self.TH = xb.num_tiles(cam0, self.cfg)
        self.T = self.TW * self.TH * self.V           # tiles of all views (tile id of view v: v T_view + t)
        d, f32, i32 = self.device, torch.float32, torch.int32
        N = self.N * self.V                           # per-(view, Gaussian) arrays, view-major
        e = lambda *s, dtype=f32: torch.empty(*s, dtype=dtype, device=d)
        # projection outputs (a1-a3)
        self.mean2d, self.conic_opac, self.rgb = e(N, 2), e(N, 4), e(N, 3)
        self.depth, self.lnv = e(N), e(N)
        self.tile_rect, self.tile_count = e(N, 4, dtype=i32), e(N, dtype=i32)
        self.flags = e(N, dtype=torch.uint8)
        self.shade_rec = e(N, 12)                            # shader data p_sd, 48 bytes per Gaussian (xpr.h)
        # binning / sort outputs (a4-a7)
        self.tile_ranges = e(self.T, 2, dtype=i32)
        # scheduling order of the tiles for the compositing kernels (xpr_config.tile_order; no effect on results)
        # default ("auto", -1): on where the heaviest tiles bound the compositing launches (64 <= T < 4096 tiles:
        # measured -4 % per step at 800x800), off for large images, where it only costs its 8 us
        self.tile_order = None
        want = cfg.get("tile_order", -1) if isinstance(cfg, dict) else -1
        if want == 1 or (want == -1 and 64 <= self.T < 4096):
            self.tile_order = torch.arange(self.T, dtype=i32, device=d)
            self.cfg.tile_order = self.tile_order.data_ptr()
        self.num_pairs = 0
        self._alloc_pairs(int(pair_capacity) if pair_capacity else max(1 << 16, 8 * N))
        # compositing outputs (a8)
        vshape = (self.V,) if self.V > 1 else ()
        self.image, self.final_T = e(*vshape, self.H, self.W, 3), e(*vshape, self.H, self.W)
        self.n_contrib = e(*vshape, self.H, self.W, dtype=i32)
        # gradients (a9, a10)
        # the compositing gradients share one allocation, in the order the library checks for, so that
        # xpr_rasterize_bwd zero-fills them with a single memset
        g2 = e(10 * N)                                     # ... | g_depth (f3) last
        self._g2, self._zeroed2d = g2, False
        self.g_mean2d, self.g_conic = g2[:2 * N].view(N, 2), g2[2 * N:5 * N].view(N, 3)
        self.g_opac, self.g_rgb, self.g_depth = g2[5 * N:6 * N], g2[6 * N:9 * N].view(N, 3), g2[9 * N:]
        if self.features:
            self.depth_img, self.alpha_img = e(*vshape, self.H, self.W), e(*vshape, self.H, self.W)
        # the parameter gradients share one allocation, in the order the library checks for (one zero-fill in xpr_project_bwd)
        N = self.N                                     # (summed over the views of a batch)
        K3 = 3 * self.K
        g4 = e((11 + K3) * N)
        self.g_means, self.g_scales = g4[:3 * N].view(N, 3), g4[3 * N:6 * N].view(N, 3)
        self.g_quats, self.g_opacities = g4[6 * N:10 * N].view(N, 4), g4[10 * N:11 * N]
        self.g_sh = g4[11 * N:].view(N, self.K, 3)
        if self.ray_eval:   # f2: shader record, per-pixel rays, record gradient
            self.ray_rec = e(N, 12)
            g3 = e(21 * N)                                 # g_ray_acc | g_opac | g_rgb | g_depth: one memset in the ray backward
            self.g_ray_acc = g3[:16 * N].view(N, 16)
            self.g_opac, self.g_rgb, self.g_depth = g3[16 * N:17 * N], g3[17 * N:20 * N].view(N, 3), g3[20 * N:]
            self.pixel_rays = e(self.H, self.W, 3)
            self.pixel_info()
            self.g_mean2d.zero_(); self.g_conic.zero_()    # the footprint carries no gradient

    def _alloc_pairs(self, cap: int):
        cap = min(int(cap), (1 << 30) - 1)
        self.pair_capacity = cap
        d = self.device
        self.keys_sorted = torch.empty(max(cap, 1), dtype=torch.int64, device=d)
        self.vals_sorted = torch.empty(max(cap, 1), dtype=torch.int32, device=d)
        ws = xb.xpr_bin_sort_workspace(self.N * self.V, cap, self.T)
        self.workspace = torch.empty(ws, dtype=torch.uint8, device=d)

    # ---- stages ------------------------------------------------------------------------------
    def project(self, means, scales, quats, opacities, sh):
        self._inputs = (means, scales, quats, opacities, sh)
        xb.xpr_project(means, scales, quats, opacities, sh, self.cam, self.cfg, self.mean2d, self.conic_opac, self.rgb,
                       self.depth, self.lnv, self.tile_rect, self.tile_count, self.flags, self.shade_rec)

    def pixel_info(self):
        xb.xpr_pixel_info(self.cam, self.pixel_rays)

    def project_ray(self):
        means, scales, quats, _, _ = self._inputs
        xb.xpr_project_ray(means, scales, quats, self.cam, self.tile_count, self.ray_rec)

    def bin_sort(self):
        self._fork_fill(2)
        while True:
            st, n = xb.xpr_bin_sort(self.depth, self.tile_rect, self.tile_count, self.cam, self.cfg,
                                    self.pair_capacity, self.keys_sorted, self.vals_sorted, self.tile_ranges,
                                    self.workspace, raise_on_capacity=False, cull_data=self._cull_data())
            if st == xb.XPR_OK:
                self.num_pairs = n
                return n
            if n >= (1 << 30):
                raise xb.XprError(st, "xpr_bin_sort (pair count exceeds 2^30)")
            self._alloc_pairs(int(n * 1.25) + 1024)   # XPR_ERR_CAPACITY: regrow and redo

    def bin_sort_async(self):
        """xpr_bin_sort without the host read-back of I (num_pairs_host = NULL): nothing in the step waits for
        the host, so the whole step can be enqueued ahead or captured in a CUDA graph.  The buffers must have
        been sized by an earlier bin_sort(); pairs_on_device() / check_capacity() read the count afterwards."""
        self._fork_fill(2)
        xb.xpr_bin_sort(self.depth, self.tile_rect, self.tile_count, self.cam, self.cfg, self.pair_capacity,
                        self.keys_sorted, self.vals_sorted, self.tile_ranges, self.workspace, sync=False,
                        cull_data=self._cull_data())

    def _cull_data(self):
        """tile-cull data p_tcd of the projection when cfg.tile_cull is set -> xpr_bin_sort_cull."""
        return (self.mean2d, self.conic_opac, self.lnv) if int(self.cfg.tile_cull) else None

    def pairs_on_device(self):
        """(I or, when it does not fit, the capacity that suffices; pairs in the sorted output) of the last bin_sort
        call, from the first 16 bytes of the workspace (synchronises)."""
        c = self.workspace[:16].view(torch.int64).tolist()
        return int(c[0]), int(c[1])

    def rows_on_device(self) -> int:
        """Number of (Gaussian, tile row) segments of the last bin_sort call (workspace bytes [24, 32))."""
        return int(self.workspace[24:32].view(torch.int64).item())

    def words_on_device(self) -> int:
        """Number of (Gaussian, supertile) words of the last bin_sort call (workspace bytes [16, 24))."""
        return int(self.workspace[16:24].view(torch.int64).item())

    def candidates_on_device(self) -> int:
        """Candidate pairs (sum of tile_count over the visible Gaussians) of the last call (workspace bytes [40, 48))."""
        return int(self.workspace[40:48].view(torch.int64).item())

    def check_capacity(self):
        cand, n = self.pairs_on_device()
        if cand > self.pair_capacity:
            raise xb.XprError(xb.XPR_ERR_CAPACITY, f"xpr_bin_sort (asynchronous): {cand} pairs > capacity {self.pair_capacity}")
        self.num_pairs = n
        return n

    def rasterize_fwd(self):
        self._fork_fill(4)      # (the parameter-gradient arrays of the previous step are cleared from here on)
        if self.ray_eval and self.features:
            xb.xpr_rasterize_ray_feat_fwd(self.cam, self.cfg, self.ray_rec, self.conic_opac, self.rgb, self.lnv, self.depth,
                                          self.pixel_rays, self.vals_sorted, self.tile_ranges, self.image, self.final_T,
                                          self.n_contrib, self.depth_img, self.alpha_img)
            return
        if self.ray_eval:
            xb.xpr_rasterize_ray_fwd(self.cam, self.cfg, self.ray_rec, self.conic_opac, self.rgb, self.lnv,
                                     self.pixel_rays, self.vals_sorted, self.tile_ranges, self.image, self.final_T,
                                     self.n_contrib)
            return
        if self.features:
            xb.xpr_rasterize_feat_fwd(self.cam, self.cfg, self.shade_rec, self.vals_sorted, self.tile_ranges, self.image,
                                      self.final_T, self.n_contrib, self.depth_img, self.alpha_img)
            return
        xb.xpr_rasterize_fwd(self.cam, self.cfg, self.shade_rec, self.vals_sorted, self.tile_ranges, self.image,
                             self.final_T, self.n_contrib)

    OVERLAP_MIN_BYTES = 32 << 20

    def _fork_fill(self, where: int):
        if self.overlap_fill != where or self._filled:
            return
        if self.N * (11 + 3 * self.K) * 4 < self.OVERLAP_MIN_BYTES:      # small scenes: the fork / join costs more than the fill
            return
        if not hasattr(self, "_side"):
            self._side = torch.cuda.Stream(device=self.device)
            self._ev_fork, self._ev_join, self._ev_join2d = torch.cuda.Event(), torch.cuda.Event(), torch.cuda.Event()
        self._ev_fork.record(torch.cuda.current_stream())      # after every earlier reader / writer of the gradient arrays
        self._side.wait_event(self._ev_fork)
        if where == 4 and not self.ray_eval:
            # the 2D gradients of the compositing backward (40 B per Gaussian) first: the backward waits for THIS event only
            with torch.cuda.stream(self._side):
                self._g2.zero_()
            self._ev_join2d.record(self._side)
            self._zeroed2d = True
        xb.xpr_project_bwd_fill(self.cfg, self.g_means, self.g_scales, self.g_quats, self.g_opacities, self.g_sh,
                                stream=self._side)
        self._ev_join.record(self._side)
        self._filled = True

    def rasterize_bwd(self, dL_dimage, dL_ddepth=None, dL_dalpha=None):
        self._feat_bwd = False
        self._fork_fill(1)
        if self.features and (dL_ddepth is not None or dL_dalpha is not None):
            z = lambda t: torch.zeros_like(self.final_T) if t is None else t
            if self.ray_eval:
                xb.xpr_rasterize_ray_feat_bwd(self.cam, self.cfg, self.ray_rec, self.conic_opac, self.rgb, self.lnv,
                                              self.depth, self.pixel_rays, self.vals_sorted, self.tile_ranges, self.final_T,
                                              self.n_contrib, dL_dimage, z(dL_ddepth), z(dL_dalpha), self.g_ray_acc,
                                              self.g_opac, self.g_rgb, self.g_depth, zero_init=True)
                self._feat_bwd = True
                return
            xb.xpr_rasterize_feat_bwd(self.cam, self.cfg, self.shade_rec, self.vals_sorted, self.tile_ranges,
                                      self.final_T, self.n_contrib, dL_dimage,
                                      z(dL_ddepth), z(dL_dalpha), self.g_mean2d, self.g_conic, self.g_opac,
                                      self.g_rgb, self.g_depth, zero_init=self._zero_init_2d())
            self._feat_bwd = True
            return
        if self.ray_eval:
            xb.xpr_rasterize_ray_bwd(self.cam, self.cfg, self.ray_rec, self.conic_opac, self.rgb, self.lnv,
                                     self.pixel_rays, self.vals_sorted, self.tile_ranges, self.final_T, self.n_contrib,
                                     dL_dimage, self.g_ray_acc, self.g_opac, self.g_rgb, zero_init=True)
            return
        xb.xpr_rasterize_bwd(self.cam, self.cfg, self.shade_rec, self.vals_sorted, self.tile_ranges, self.final_T,
                             self.n_contrib, dL_dimage, self.g_mean2d, self.g_conic, self.g_opac, self.g_rgb,
                             zero_init=self._zero_init_2d())

    def _zero_init_2d(self) -> bool:
        """False when the 2D gradient arrays were already cleared on the side stream (overlap_fill 4): the backward then
        waits for that memset instead of issuing its own."""
        if not self._zeroed2d:
            return True
        self._zeroed2d = False
        torch.cuda.current_stream().wait_event(self._ev_join2d)
        return False

    def can_fuse_loss(self) -> bool:
        return self.fuse_loss and not self.ray_eval and not self.features

    def rasterize_bwd_loss(self, target, loss: str):
        """xpr_loss_grad + xpr_rasterize_bwd in one launch (the loss gradient is formed in the kernel's prologue)."""
        self._feat_bwd = False
        self._fork_fill(1)
        xb.xpr_rasterize_bwd_loss(self.cam, self.cfg, self.shade_rec, self.vals_sorted, self.tile_ranges, self.image,
                                  self.final_T, self.n_contrib, loss, target, self.g_mean2d, self.g_conic, self.g_opac,
                                  self.g_rgb, zero_init=self._zero_init_2d())

    # ---- N-channel features (f3): replay of the finished colour pass ---------------------------
    def rasterize_featn_fwd(self, feat, feat_img=None):
        """feat [N,C] -> feat_img [H,W,C] = sum_k feat[g_k,:] alpha_k T_k (call after rasterize_fwd)."""
        if self.ray_eval:
            raise ValueError("xpr: N-channel features are built for the 2D evaluation")
        if feat_img is None:
            feat_img = torch.empty(self.H, self.W, feat.shape[1], dtype=torch.float32, device=self.device)
        xb.xpr_rasterize_featn_fwd(self.cam, self.cfg, self.mean2d, self.conic_opac, self.lnv, feat, self.vals_sorted,
                                   self.tile_ranges, self.n_contrib, feat_img)
        return feat_img

    def rasterize_featn_bwd(self, feat, dL_dfeat, g_feat=None, first: bool = False):
        """Adds the feature part of the compositing gradients (call between rasterize_bwd and project_bwd; first=True
        when no colour backward ran: the geometric gradients are then zero-filled here); returns g_feat [N,C]."""
        if g_feat is None:
            g_feat = torch.empty_like(feat)
        xb.xpr_rasterize_featn_bwd(self.cam, self.cfg, self.mean2d, self.conic_opac, self.lnv, feat, self.vals_sorted,
                                   self.tile_ranges, self.final_T, self.n_contrib, dL_dfeat, self.g_mean2d, self.g_conic,
                                   self.g_opac, g_feat, zero_init=3 if first else 2)
        if first:
            self.g_rgb.zero_()
            self._feat_bwd = False
        return g_feat

    def project_bwd(self):
        means, scales, quats, opacities, sh = self._inputs
        filled, self._filled = self._filled, False
        if filled:
            torch.cuda.current_stream().wait_event(self._ev_join)
        xb.xpr_project_bwd(means, scales, quats, opacities, sh, self.cam, self.cfg, self.tile_count, self.flags,
                           self.g_mean2d, self.g_conic, self.g_opac, self.g_rgb, self.g_means, self.g_scales,
                           self.g_quats, self.g_opacities, self.g_sh, filled=filled)
        if self.ray_eval:
            xb.xpr_ray_bwd(means, scales, quats, self.cam, self.tile_count, self.g_ray_acc, self.g_means,
                           self.g_scales, self.g_quats)
        if getattr(self, "_feat_bwd", False):
            if self.V > 1:      # z of view v is (W_v mu + t_v)_z: the call ADDS, so the views accumulate one after the other
                N = self.N
                for v in range(self.V):
                    xb.xpr_depth_bwd(self.cam[v], self.tile_count[v * N:(v + 1) * N], self.g_depth[v * N:(v + 1) * N],
                                     self.g_means)
            else:
                xb.xpr_depth_bwd(self.cam, self.tile_count, self.g_depth, self.g_means)

    # ---- whole passes -------------------------------------------------------------------------
    def forward(self, means, scales, quats, opacities, sh):
        self.project(means, scales, quats, opacities, sh)
        if self.ray_eval:
            self.project_ray()
        self.bin_sort()
        self.rasterize_fwd()
        return self.image

    def backward(self, dL_dimage, dL_ddepth=None, dL_dalpha=None):
        self.rasterize_bwd(dL_dimage, dL_ddepth, dL_dalpha)
        self.project_bwd()
        return dict(g_means=self.g_means, g_scales=self.g_scales, g_quats=self.g_quats,
                    g_opacities=self.g_opacities, g_sh=self.g_sh)

    def step_async(self, means, scales, quats, opacities, sh, target, loss: str, pixel_info: bool = False):
        """One training step (forward, dL/dimage of `loss` against `target`, backward) enqueued on the current
        stream without any host read-back: xpr_bin_sort runs with num_pairs_host = NULL.  The pair buffers must
        have been sized by an earlier forward(); call check_capacity() once the stream has run."""
        if self._dL is None:
            self._dL = torch.empty_like(self.image)
        self.project(means, scales, quats, opacities, sh)
        if self.ray_eval:
            if pixel_info:
                self.pixel_info()
            self.project_ray()
        self.bin_sort_async()
        self.rasterize_fwd()
        if self.can_fuse_loss():
            self.rasterize_bwd_loss(target, loss)
        else:
            xb.xpr_loss_grad(loss, self.image, target, self._dL)
            self.rasterize_bwd(self._dL, *(self.feature_grads or (None, None)))
        self.project_bwd()

    def capture_step(self, means, scales, quats, opacities, sh, target, loss: str, pixel_info: bool = False):
        """step_async() captured once into a CUDA graph (nothing on the path waits for the host, so the whole step
        is capturable); graph.replay() then runs a step on the same buffers with no per-launch host work."""
        side = torch.cuda.Stream(self.device)
        side.wait_stream(torch.cuda.current_stream(self.device))
        with torch.cuda.stream(side):                    # warm-up outside the capture (lazy module loading)
            self.step_async(means, scales, quats, opacities, sh, target, loss, pixel_info)
        torch.cuda.current_stream(self.device).wait_stream(side)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            self.step_async(means, scales, quats, opacities, sh, target, loss, pixel_info)
        return graph


def scene_to_device(scene, device="cuda:0"):
    """Upload a scenes.Scene's parameter arrays; returns (means, scales, quats, opacities, sh)."""
    t = lambda a: torch.from_numpy(a).to(device).contiguous()
    return t(scene.means), t(scene.scales), t(scene.quats), t(scene.opacities), t(scene.sh)


class LinPrimPipeline:
    """XPR-LinPrim (PAPER A.1.3): xpr_lin_project -> xpr_bin_sort_lin -> xpr_lin_rasterize_fwd ->
    [loss outside] -> xpr_lin_rasterize_bwd -> xpr_lin_project_bwd.  Buffers and call order only, like SplatPipeline;
    one pinhole view."""

    def __init__(self, N: int, cam, cfg: dict, pair_capacity: int | None = None, device="cuda:0"):
        self.N = int(N)
        self.device = torch.device(device)
        self.cam = cam if isinstance(cam, xb.XprCamera) else xb.make_camera(cam)
        self.cfg = cfg if isinstance(cfg, xb.XprConfig) else xb.make_config(cfg)
        self.W, self.H = int(self.cam.width), int(self.cam.height)
        self.TW, self.TH = xb.num_tiles(self.cam, self.cfg)
        self.T = self.TW * self.TH
        d, f32, i32 = self.device, torch.float32, torch.int32
        e = lambda *s, dtype=f32: torch.empty(*s, dtype=dtype, device=d)
        self.lin_rec, self.depth = e(self.N, 20), e(self.N)
        self.tile_rect, self.tile_count = e(self.N, 4, dtype=i32), e(self.N, dtype=i32)
        self.tile_ranges = e(self.T, 2, dtype=i32)
        self.image, self.final_T = e(self.H, self.W, 3), e(self.H, self.W)
        self.n_contrib = e(self.H, self.W, dtype=i32)
        self.K = (int(self.cfg.sh_degree) + 1) ** 2
        self.g_lin_rec = e(self.N, 20)
        self.g_means, self.g_scales, self.g_quats = e(self.N, 3), e(self.N, 3), e(self.N, 4)
        self.g_opacities, self.g_sh = e(self.N), e(self.N, self.K, 3)
        self.num_pairs = 0
        self._alloc_pairs(int(pair_capacity) if pair_capacity else max(1 << 16, 8 * self.N))

    _alloc_pairs = SplatPipeline._alloc_pairs
    V = 1

    def project(self, means, scales, quats, opacities, sh):
        self._inputs = (means, scales, quats, opacities, sh)
        xb.xpr_lin_project(means, scales, quats, opacities, sh, self.cam, self.cfg, self.lin_rec, self.depth,
                           self.tile_rect, self.tile_count)

    def bin_sort(self):
        while True:
            st, n = xb.xpr_bin_sort(self.depth, self.tile_rect, self.tile_count, self.cam, self.cfg,
                                    self.pair_capacity, self.keys_sorted, self.vals_sorted, self.tile_ranges,
                                    self.workspace, raise_on_capacity=False, lin_rec=self.lin_rec)
            if st == xb.XPR_OK:
                self.num_pairs = n
                return n
            if n >= (1 << 30):
                raise xb.XprError(st, "xpr_bin_sort_lin (pair count exceeds 2^30)")
            self._alloc_pairs(int(n * 1.25) + 1024)

    def rasterize_fwd(self):
        xb.xpr_lin_rasterize_fwd(self.cam, self.cfg, self.lin_rec, self.vals_sorted, self.tile_ranges, self.image,
                                 self.final_T, self.n_contrib)

    def forward(self, means, scales, quats, opacities, sh):
        self.project(means, scales, quats, opacities, sh)
        self.bin_sort()
        self.rasterize_fwd()
        return self.image

    def bin_sort_async(self):
        """xpr_bin_sort_lin without the host read-back (buffers sized by an earlier bin_sort())."""
        xb.xpr_bin_sort(self.depth, self.tile_rect, self.tile_count, self.cam, self.cfg, self.pair_capacity,
                        self.keys_sorted, self.vals_sorted, self.tile_ranges, self.workspace, sync=False,
                        lin_rec=self.lin_rec)

    def rasterize_bwd(self, dL_dimage):
        xb.xpr_lin_rasterize_bwd(self.cam, self.cfg, self.lin_rec, self.vals_sorted, self.tile_ranges, self.final_T,
                                 self.n_contrib, dL_dimage, self.g_lin_rec)

    def project_bwd(self):
        xb.xpr_lin_project_bwd(*self._inputs, self.cam, self.cfg, self.tile_count, self.lin_rec, self.g_lin_rec,
                               self.g_means, self.g_scales, self.g_quats, self.g_opacities, self.g_sh)

    def backward(self, dL_dimage):
        self.rasterize_bwd(dL_dimage)
        self.project_bwd()
