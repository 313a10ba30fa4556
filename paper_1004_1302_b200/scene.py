"""Convenience layer over the binding: device residency of a particle set and one-call renders.

Argument marshalling and memory management only (PyTorch owns device memory and streams);
every step of the path runs in libsplotch_b200.so.
"""
from __future__ import annotations

from typing import Optional

import numpy as np
import torch

from . import binding as B


def _camera_struct(cam) -> B.splotch_camera:
    return B.make_camera(cam.eye, cam.lookat, cam.up, cam.fov_deg, cam.width, cam.height)


class Scene:
    """A particle set resident in HBM plus its colour tables and parameters.

    `w` is any object with the fields of workloads.Workload (numpy arrays x, y, z, r, I, colval,
    optional uint8 type, lut_e/lut_a of shape (n_types, n_entries, 3), brightness lists, mode,
    support_f, z_near, cameras)."""

    def __init__(self, w, device: str = "cuda:0", resident: bool = True):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1004_1302_b200 needs a CUDA device: there is no CPU fallback")
        B.library_path()   # fail loudly if the extension is missing
        self.device = torch.device(device)
        self.w = w
        self.n = int(w.n)
        self.n_types, self.n_entries = int(w.lut_e.shape[0]), int(w.lut_e.shape[1])
        self._host = {k: np.ascontiguousarray(getattr(w, k), np.float32) for k in ("x", "y", "z", "r", "I", "colval")}
        self._host_type = None if w.type is None else np.ascontiguousarray(w.type, np.uint8)
        vec = getattr(w, "vec", None)       # optional (n, 3) vector colouring
        self._host_vec = None if vec is None else [np.ascontiguousarray(np.asarray(vec, np.float32)[:, k]) for k in range(3)]
        self._host_lut_e = np.ascontiguousarray(w.lut_e, np.float32)
        self._host_lut_a = None if w.lut_a is None else np.ascontiguousarray(w.lut_a, np.float32)
        self.d = {}
        self.workspace: Optional[torch.Tensor] = None
        self.max_pairs = 0
        self._counted = set()     # (camera, mode) keys whose pair count render_batch has already checked against max_pairs
        self.tensor = None        # additive mode: None = library decides, True = SPLOTCH_FORCE_TENSOR, False = SPLOTCH_NO_TENSOR
        if resident:
            self.upload()

    # ---- device residency ----------------------------------------------------------------
    def upload(self) -> None:
        with torch.cuda.device(self.device):
            for k, a in self._host.items():
                self.d[k] = torch.from_numpy(a).to(self.device)
            self.d["type"] = None if self._host_type is None else torch.from_numpy(self._host_type).to(self.device)
            self.d["vec"] = None if self._host_vec is None else [torch.from_numpy(a).to(self.device) for a in self._host_vec]
            self.d["lut_e"] = torch.from_numpy(self._host_lut_e).to(self.device)
            self.d["lut_a"] = None if self._host_lut_a is None else torch.from_numpy(self._host_lut_a).to(self.device)
            torch.cuda.synchronize(self.device)

    def particles(self) -> B.splotch_particles:
        d = self.d
        return B.make_particles(d["x"], d["y"], d["z"], d["r"], d["I"], d["colval"], d["type"], d["vec"])

    def colormap(self) -> B.splotch_colormap:
        return B.make_colormap(self.d["lut_e"], self.d["lut_a"], self.n_entries, self.n_types)

    def params(self, mode: Optional[int] = None, raw: bool = False) -> B.splotch_params:
        w = self.w
        flags = (B.SPLOTCH_RAW_SUM if raw else 0) | (0 if self.tensor is None else B.SPLOTCH_FORCE_TENSOR if self.tensor else B.SPLOTCH_NO_TENSOR)
        return B.make_params(w.brightness, w.abs_brightness, w.mode if mode is None else mode, w.support_f, w.z_near, flags)

    def _alloc(self, nbytes: int) -> torch.Tensor:
        return torch.empty(int(nbytes) + 256, dtype=torch.uint8, device=self.device)

    def _cam_key(self, cam, mode):
        return (tuple(cam.eye), tuple(cam.lookat), tuple(cam.up), float(cam.fov_deg), int(cam.width), int(cam.height),
                self.w.mode if mode is None else mode)

    @staticmethod
    def _aligned(t: torch.Tensor) -> int:
        return (t.data_ptr() + 255) // 256 * 256

    # ---- sizing ---------------------------------------------------------------------------
    def count_pairs(self, cam=None, mode: Optional[int] = None):
        """(pairs, visible) for a camera; synchronises."""
        cam = cam or self.w.camera
        cs, ps = _camera_struct(cam), self.params(mode)
        nbytes = B.splotch_workspace_bytes(self.n, cs, ps, 0)
        ws = self._alloc(nbytes)
        return B.splotch_count_pairs(self.particles(), self.n, cs, self.colormap(), ps, self._aligned(ws), nbytes)

    def reserve(self, cam=None, mode: Optional[int] = None, max_pairs: Optional[int] = None, slack: float = 1.02) -> int:
        """Size and allocate the workspace for `cam` (or for an explicit max_pairs)."""
        cam = cam or self.w.camera
        if max_pairs is None:
            pairs, _ = self.count_pairs(cam, mode)
            max_pairs = int(pairs * slack) + 1024
        cs, ps = _camera_struct(cam), self.params(mode)
        nbytes = B.splotch_workspace_bytes(self.n, cs, ps, max_pairs)
        if self.workspace is None or self.workspace.numel() < nbytes + 256:
            self.workspace = None
            self.workspace = self._alloc(nbytes)
        self.max_pairs = int(max_pairs)
        return nbytes

    # ---- the render call ------------------------------------------------------------------
    def render(self, cam=None, mode: Optional[int] = None, raw: bool = False, out: Optional[torch.Tensor] = None,
               check: bool = True) -> torch.Tensor:
        """One splotch_render on the current stream.  Returns a float32 (H, W, 3) CUDA tensor."""
        cam = cam or self.w.camera
        cs, ps = _camera_struct(cam), self.params(mode, raw)
        nbytes = B.splotch_workspace_bytes(self.n, cs, ps, self.max_pairs) if self.workspace is not None else None
        if self.workspace is None or self.workspace.numel() < nbytes + 256:
            nbytes = self.reserve(cam, mode)
        if out is None:
            out = torch.empty((cam.height, cam.width, 3), dtype=torch.float32, device=self.device)
        B.splotch_render(self.particles(), self.n, cs, self.colormap(), ps, out, self._aligned(self.workspace),
                         self.workspace.numel() - 256, self.max_pairs)
        if check:
            status, _, pairs = B.splotch_workspace_status(self._aligned(self.workspace))
            if status != B.SPLOTCH_OK:
                raise B.SplotchError(f"splotch_render (scene needs {pairs} pairs, max_pairs={self.max_pairs})", status)
        return out

    def render_batch(self, cams=None, mode: Optional[int] = None, raw: bool = False, out: Optional[torch.Tensor] = None,
                     check: bool = True):
        """One splotch_render_batch over `cams` (default: every camera of the workload: the orbit).  Returns
        (images (K, H, W, 3) float32 CUDA tensor, frame_status (K, 4) int64 CUDA tensor: status, visible, pairs, 0).
        The workspace is sized once for the largest pair count over the cameras."""
        cams = list(self.w.cameras if cams is None else cams)
        K = len(cams)
        cs = [_camera_struct(c) for c in cams]
        ps = self.params(mode, raw)
        # A workspace reserved earlier for ONE camera may be too small for another camera of the batch: the pair counts of
        # cameras this scene has not counted yet are taken once (synchronising) and the workspace grown if one needs more.
        # Cameras already counted cost nothing, so a steady orbit loop, or a caller that lowers max_pairs on purpose, is
        # left alone.
        new = [c for c in cams if self._cam_key(c, mode) not in self._counted]
        if new or self.workspace is None:
            worst = max(self.count_pairs(c, mode)[0] for c in new) if new else 0
            self._counted.update(self._cam_key(c, mode) for c in new)
            need = B.splotch_workspace_bytes(self.n, cs[0], ps, max(self.max_pairs, worst)) if K else 0
            if self.workspace is None or self.max_pairs < worst or self.workspace.numel() < need + 256:
                self.reserve(cams[0] if K else None, mode, max_pairs=max(self.max_pairs, worst + 1024))
        H, W = (cams[0].height, cams[0].width) if K else (0, 0)
        if out is None:
            out = torch.empty((K, H, W, 3), dtype=torch.float32, device=self.device)
        status = torch.zeros((max(K, 1), 4), dtype=torch.int64, device=self.device)
        B.splotch_render_batch(self.particles(), self.n, cs, self.colormap(), ps, out, status, self._aligned(self.workspace),
                               self.workspace.numel() - 256, self.max_pairs)
        if check:
            bad = [(k, int(r[2])) for k, r in enumerate(status[:K].cpu().tolist()) if r[0] != B.SPLOTCH_OK]
            if bad:
                raise B.SplotchError(f"splotch_render_batch (frames {bad} need more than max_pairs={self.max_pairs})",
                                     B.SPLOTCH_ERR_WORKSPACE)
        return out, status[:K]

    def stats(self, cam=None, mode: Optional[int] = None, bin_shift: int = 6):
        """(visible, pairs at bin_shift, pixel updates U); synchronises."""
        cam = cam or self.w.camera
        cs, ps = _camera_struct(cam), self.params(mode)
        nbytes = B.splotch_debug_workspace_bytes(self.n, cs, ps, bin_shift, 0)
        ws = self._alloc(nbytes)
        return B.splotch_debug_stats(self.particles(), self.n, cs, self.colormap(), ps, self._aligned(ws), nbytes, bin_shift)

    def tensor_stats(self, cam=None):
        """(updates the tensor-core rasteriser performs, the library's choice 0/1, estimated share); synchronises."""
        cam = cam or self.w.camera
        cs, ps = _camera_struct(cam), self.params(0)
        nbytes = B.splotch_debug_workspace_bytes(self.n, cs, ps, 6, 0)
        ws = self._alloc(nbytes)
        return B.splotch_debug_tensor_stats(self.particles(), self.n, cs, self.colormap(), ps, self._aligned(ws), nbytes)

    # ---- end to end with host buffers ---------------------------------------------------------
    def host_buffers(self, pinned: bool = True):
        """Pinned host copies of the inputs and a pinned output image for render_host."""
        def pin(a):
            t = torch.from_numpy(a)
            return t.pin_memory() if pinned else t
        hb = {k: pin(a) for k, a in self._host.items()}
        hb["type"] = None if self._host_type is None else pin(self._host_type)
        hb["lut_e"] = pin(self._host_lut_e)
        hb["lut_a"] = None if self._host_lut_a is None else pin(self._host_lut_a)
        return hb

    def render_host(self, hb, cam=None, mode: Optional[int] = None, out_host: Optional[torch.Tensor] = None,
                    max_pairs: Optional[int] = None, workspace: Optional[torch.Tensor] = None):
        """splotch_render_host: H2D copies + render + D2H copy + sync inside the library call."""
        cam = cam or self.w.camera
        cs, ps = _camera_struct(cam), self.params(mode)
        max_pairs = self.max_pairs if max_pairs is None else max_pairs
        ph = B.make_particles(hb["x"], hb["y"], hb["z"], hb["r"], hb["I"], hb["colval"], hb["type"])
        cmh = B.make_colormap(hb["lut_e"], hb["lut_a"], self.n_entries, self.n_types)
        nbytes = B.splotch_workspace_bytes_host(self.n, cs, cmh, ps, max_pairs)
        if workspace is None:
            workspace = self._alloc(nbytes)
        if out_host is None:
            out_host = torch.empty((cam.height, cam.width, 3), dtype=torch.float32).pin_memory()
        B.splotch_render_host(ph, self.n, cs, cmh, ps, out_host, self._aligned(workspace), nbytes, max_pairs)
        return out_host, workspace

    def render_host_pipelined(self, hb, n_frames: int, cam=None, mode: Optional[int] = None, max_pairs: Optional[int] = None,
                              depth: int = 2):
        """`n_frames` end-to-end frames (H2D of the inputs + render + D2H of the image, every frame) through
        splotch_render_host_async with `depth` frames in flight: frame k + 1 is copied in while frame k is rasterised.
        Each slot has its own stream, device workspace and pinned output image.  Returns the list of output images of
        the last `depth` frames (pinned host tensors).  Synchronises at the end; raises if any frame failed."""
        cam = cam or self.w.camera
        cs, ps = _camera_struct(cam), self.params(mode)
        max_pairs = self.max_pairs if max_pairs is None else max_pairs
        ph = B.make_particles(hb["x"], hb["y"], hb["z"], hb["r"], hb["I"], hb["colval"], hb["type"])
        cmh = B.make_colormap(hb["lut_e"], hb["lut_a"], self.n_entries, self.n_types)
        nbytes = B.splotch_workspace_bytes_host(self.n, cs, cmh, ps, max_pairs)
        # keyed on the image shape too: a camera with width and height swapped needs the same bytes but another (H, W)
        key = (cam.height, cam.width, nbytes, depth)
        if getattr(self, "_pipe", None) is None or self._pipe["key"] != key:
            self._pipe = dict(key=key, nbytes=nbytes, ws=[self._alloc(nbytes) for _ in range(depth)],
                              streams=[torch.cuda.Stream(self.device) for _ in range(depth)],
                              out=[torch.empty((cam.height, cam.width, 3), dtype=torch.float32).pin_memory() for _ in range(depth)],
                              busy=[False] * depth)
        P = self._pipe

        def finish(slot):
            if P["busy"][slot]:
                status, _, pairs = B.splotch_workspace_status(self._aligned(P["ws"][slot]), P["streams"][slot])
                P["busy"][slot] = False
                if status != B.SPLOTCH_OK:
                    raise B.SplotchError(f"splotch_render_host_async (scene needs {pairs} pairs, max_pairs={max_pairs})", status)

        for k in range(n_frames):
            slot = k % depth
            finish(slot)                      # the slot's previous frame has left its stream: its buffers are free again
            B.splotch_render_host_async(ph, self.n, cs, cmh, ps, P["out"][slot], self._aligned(P["ws"][slot]), nbytes, max_pairs,
                                        P["streams"][slot])
            P["busy"][slot] = True
        for slot in range(depth):
            finish(slot)
        return P["out"]

    def h2d_bytes(self) -> int:
        lut = self._host_lut_e.nbytes + (0 if self._host_lut_a is None else self._host_lut_a.nbytes)
        return self.n * (24 + (0 if self._host_type is None else 1)) + lut
