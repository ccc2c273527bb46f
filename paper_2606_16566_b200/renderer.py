"""Renderer: owns the device copies of a scene, the output buffers and the workspace; one call = one frame.

This is the public Python API (the call a user makes).  It only allocates tensors and forwards to
binding.gs_render -- no arithmetic of the method lives here.
"""
from __future__ import annotations

from types import SimpleNamespace

import numpy as np
import torch

from . import binding

_SCENE_ARRAYS = ("means3D", "scales", "rotations", "opacities", "sh")


class Renderer:
    def __init__(self, P: int, W: int, H: int, max_dup: int, device="cuda:0", count_contrib: bool = True, graph=None):
        """graph: replay the frame's launch sequence as a CUDA graph (include/gs.h: gs_set_graph); None = for scenes of up to
        2^21 Gaussians, whose frames are launch-chain-bound."""
        self.P, self.W, self.H = int(P), int(W), int(H)
        self.graph = (self.P <= (1 << 21)) if graph is None else bool(graph)
        self.device = torch.device(device)
        self.gx, self.gy = (W + 15) // 16, (H + 15) // 16
        self.max_dup = int(max_dup)
        nbytes = binding.gs_workspace_bytes(P, W, H, max_dup)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        binding.gs_set_workspace_option(self.workspace, binding.GS_OPT_GRAPH, 1 if self.graph else 0)
        self.out_rgb = torch.empty((3, H, W), dtype=torch.float32, device=self.device)
        self.out_final_T = torch.empty((H, W), dtype=torch.float32, device=self.device)
        self.out_tile_counts = torch.empty((self.gy * self.gx,), dtype=torch.int32, device=self.device)
        self.out_n_contrib = torch.empty((H, W), dtype=torch.int32, device=self.device) if count_contrib else None
        self.scene = None
        self._pinned = None   # two pinned host staging sets of the scene arrays, allocated on first use
        self._pinned_read = None
        self._host_rgb = None
        self._ring = None     # render_to_host(): two device images, a copy stream and the events that order them
        self._lanes = None    # render_batch(): per-lane stream, workspace and outputs
        self._options = {}    # set_option(): per-workspace switches of this Renderer, applied to every lane's workspace
        self._copy_stream = None
        self._standby = None  # upload_async(): second set of scene buffers, upload stream and its events
        self._upload_stream = None

    # ---- host -> device ---------------------------------------------------------------------------------------------
    @staticmethod
    def pin_scene(scene):
        """A copy of `scene` whose arrays are pinned torch tensors: upload() / upload_async() copy from those directly
        (no staging pass).  The caller must not modify them while a copy is in flight."""
        out = SimpleNamespace(sh_degree=int(scene.sh_degree), bg=np.array(scene.bg, dtype=np.float32), cameras=getattr(scene, "cameras", None))
        for n in _SCENE_ARRAYS:
            setattr(out, n, torch.from_numpy(np.array(getattr(scene, n), dtype=np.float32, order="C")).pin_memory())
        return out

    def _stage_to_pinned(self, scene, k: int):
        """Host arrays of `scene` as pinned tensors: the scene's own tensors when they are pinned already, else pinned
        staging set k (allocated on first use), filled after the host -> device copy that last read that set has
        finished.  Checks P and the array shapes.  Returns (dict of pinned tensors, bytes)."""
        if int(scene.means3D.shape[0]) != self.P:
            raise ValueError("scene has %d Gaussians, this Renderer was built for %d" % (scene.means3D.shape[0], self.P))
        if self._pinned is None:
            self._pinned = [None, None]
            self._pinned_read = [torch.cuda.Event(), torch.cuda.Event()]
        if all(isinstance(getattr(scene, n), torch.Tensor) and getattr(scene, n).is_pinned() for n in _SCENE_ARRAYS):
            src = {n: getattr(scene, n) for n in _SCENE_ARRAYS}
            for n, t in src.items():
                if t.dtype != torch.float32 or not t.is_contiguous() or (self.scene is not None and tuple(t.shape) != tuple(self.scene[n].shape)):
                    raise ValueError("%s must be a contiguous float32 tensor of the shape this Renderer was sized for" % n)
            return src, sum(t.numel() * 4 for t in src.values())
        if self._pinned[k] is None:
            self._pinned[k] = {n: torch.empty(tuple(np.shape(getattr(scene, n))), dtype=torch.float32).pin_memory()
                               for n in _SCENE_ARRAYS}
        else:
            self._pinned_read[k].synchronize()      # the previous copy out of this staging set has completed
        nbytes = 0
        for n in _SCENE_ARRAYS:
            src = np.ascontiguousarray(getattr(scene, n), dtype=np.float32)
            dst = self._pinned[k][n]
            if tuple(src.shape) != tuple(dst.shape):
                raise ValueError("%s has shape %s, this Renderer was sized for %s" % (n, src.shape, tuple(dst.shape)))
            dst.numpy()[...] = src
            nbytes += src.nbytes
        return self._pinned[k], nbytes

    def _scene_meta(self, scene):
        return int(scene.sh_degree), np.array(scene.bg, dtype=np.float32)

    def upload(self, scene) -> int:
        """Host (numpy) scene -> device tensors, every call: the arrays are staged into pinned memory and copied
        asynchronously on the current stream; sh_degree and bg follow the scene.  Staging and device buffers are
        allocated on the first call and reused.  Returns the bytes copied host -> device."""
        src, nbytes = self._stage_to_pinned(scene, 0)
        deg, bg = self._scene_meta(scene)
        if self.scene is None:
            self.scene = {n: torch.empty_like(t, device=self.device) for n, t in src.items()}
        for n in _SCENE_ARRAYS:
            self.scene[n].copy_(src[n], non_blocking=True)
        self._pinned_read[0].record(torch.cuda.current_stream(self.device))
        self.scene["sh_degree"], self.scene["bg"] = deg, bg
        return nbytes

    def upload_async(self, scene) -> int:
        """Host -> device copy of `scene` into the STANDBY set of device buffers, on an upload stream: it overlaps the
        frames that are being rendered from the active set (PCIe is full duplex: the images of those frames travel the
        other way).  Two pinned staging sets are used alternately, so the host-side staging of one upload never
        overwrites memory a previous copy still reads.  activate_uploaded() makes the new set (and the scene's
        sh_degree / bg) the active one.  Returns the bytes copied."""
        if self.scene is None:
            self.upload(scene)                 # first use: allocates the first device set
        if self._standby is None:
            self._standby = {n: torch.empty_like(self.scene[n]) for n in _SCENE_ARRAYS}
            self._upload_stream = torch.cuda.Stream(device=self.device)
            self._uploaded, self._released = torch.cuda.Event(), torch.cuda.Event()
            self._released.record(torch.cuda.current_stream(self.device))
            self._async_k = 0
        self._async_k ^= 1
        k = self._async_k
        src, nbytes = self._stage_to_pinned(scene, k)
        self._standby_meta = self._scene_meta(scene)
        up = self._upload_stream
        up.wait_event(self._released)          # the frames that read the standby set (two activations ago) are done
        with torch.cuda.stream(up):
            for n in _SCENE_ARRAYS:
                self._standby[n].copy_(src[n], non_blocking=True)
        self._pinned_read[k].record(up)
        self._uploaded.record(up)
        return nbytes

    def activate_uploaded(self) -> None:
        """Later renders (enqueued on the current stream or forked from it) read the set upload_async() filled."""
        main = torch.cuda.current_stream(self.device)
        self._released.record(main)            # everything enqueued so far read the old active set
        main.wait_event(self._uploaded)
        old = {n: self.scene[n] for n in _SCENE_ARRAYS}
        for n in _SCENE_ARRAYS:
            self.scene[n] = self._standby[n]
        self._standby = old
        self.scene["sh_degree"], self.scene["bg"] = self._standby_meta

    def render(self, cam, stream=None, count_contrib: bool = True, out_rgb=None) -> None:
        s = self.scene
        if self._lanes and self._lanes[0]["render_stream"]:   # render_batch left lane 0 (this workspace) on the render stream
            binding.gs_set_workspace_option(self.workspace, binding.GS_OPT_RENDER_STREAM, 0)
            self._lanes[0]["render_stream"] = False
        binding.gs_render(s["means3D"], s["scales"], s["rotations"], s["opacities"], s["sh"], s["sh_degree"],
                          cam.viewmatrix, cam.projmatrix, cam.fx, cam.fy, cam.W, cam.H, s["bg"],
                          self.out_rgb if out_rgb is None else out_rgb,
                          self.out_final_T, self.out_tile_counts, self.out_n_contrib if count_contrib else None,
                          self.workspace, stream)

    def render_to_host(self, cam, slot: int = 0, n_slots: int = 1, count_contrib: bool = False) -> torch.Tensor:
        """Render one frame and copy its RGB image to pinned host slot `slot`, with the copy of frame k overlapping the
        render of frame k+1: two device images used alternately, the device -> host copy on a second stream, events in
        both directions.  Returns the host tensor (valid after synchronize_readback())."""
        if self._host_rgb is None or self._host_rgb.shape[0] < n_slots:
            self._host_rgb = torch.empty((n_slots, 3, self.H, self.W), dtype=torch.float32).pin_memory()
        if self._ring is None:
            self._ring = dict(img=[self.out_rgb, torch.empty_like(self.out_rgb)], k=0,
                              copy_stream=torch.cuda.Stream(device=self.device),
                              rendered=[torch.cuda.Event(), torch.cuda.Event()], copied=[torch.cuda.Event(), torch.cuda.Event()],
                              used=[False, False])
        rg = self._ring
        b = rg["k"] & 1
        rg["k"] += 1
        main = torch.cuda.current_stream(self.device)
        if rg["used"][b]:
            main.wait_event(rg["copied"][b])          # the image rendered two frames ago has left this buffer
        self.render(cam, count_contrib=count_contrib, out_rgb=rg["img"][b])
        rg["rendered"][b].record(main)
        with torch.cuda.stream(rg["copy_stream"]):
            rg["copy_stream"].wait_event(rg["rendered"][b])
            self._host_rgb[slot].copy_(rg["img"][b], non_blocking=True)
            rg["copied"][b].record(rg["copy_stream"])
        rg["used"][b] = True
        return self._host_rgb[slot]

    # ---- several frames in flight ---------------------------------------------------------------------------------
    def set_option(self, option: int, value: int) -> None:
        """Per-workspace switch (binding.GS_OPT_*; -1 = follow the process-wide setter) for EVERY workspace of this Renderer:
        its own and those of the lanes render_batch uses, present and future."""
        self._options[int(option)] = int(value)
        binding.gs_set_workspace_option(self.workspace, option, value)
        for ln in (self._lanes or [])[1:]:
            binding.gs_set_workspace_option(ln["workspace"], option, value)

    def _lane(self, k: int):
        """Lane k: its own stream, workspace and output buffers (lane 0 = this Renderer's own buffers, on its own
        stream too, so that the caller's stream only forks and joins)."""
        if self._lanes is None:
            self._lanes = []
        while len(self._lanes) <= k:
            first = len(self._lanes) == 0
            ln = dict(stream=torch.cuda.Stream(device=self.device, priority=-1),   # above the library's render stream
                      workspace=self.workspace if first else torch.empty_like(self.workspace),
                      out_rgb=self.out_rgb if first else torch.empty_like(self.out_rgb),
                      out_final_T=self.out_final_T if first else torch.empty_like(self.out_final_T),
                      out_tile_counts=self.out_tile_counts if first else torch.empty_like(self.out_tile_counts),
                      done=torch.cuda.Event(), copied=torch.cuda.Event(), copy_pending=False, render_stream=False)
            if not first:
                binding.gs_set_workspace_option(ln["workspace"], binding.GS_OPT_GRAPH, 1 if self.graph else 0)
                for opt, val in self._options.items():       # the switches of this Renderer hold for all its workspaces
                    binding.gs_set_workspace_option(ln["workspace"], opt, val)
            self._lanes.append(ln)
        return self._lanes[k]

    def render_batch(self, cams, lanes: int = 3, out_rgb=None, to_host: bool = False):
        """Render every camera of `cams`, `lanes` frames in flight: frame i runs on lane i % lanes (own stream, own
        workspace).  Frames are independent, so the small, latency-bound kernels of one frame's binning fill the GPU
        under the render kernel of another; every frame is computed by exactly the same launches as render().
          out_rgb   optional device tensor [len(cams), 3, H, W]: frame i writes its image there (otherwise the image of
                    frame i stays in lane i % lanes until frame i + lanes overwrites it);
          to_host   copy every image to pinned host memory on a copy stream, overlapping the later frames; returns the
                    host tensor [len(cams), 3, H, W] (valid when this call returns control to the current stream's
                    order: the current stream waits for all lanes and copies).
        The current stream is joined to all lanes before returning, so later work on it sees the results."""
        n = len(cams)
        lanes = max(1, min(int(lanes), n))
        if lanes == 1 and not to_host:      # one frame in flight: the caller's stream, no forks, no events
            for i, cam in enumerate(cams):
                self.render(cam, count_contrib=False, out_rgb=None if out_rgb is None else out_rgb[i])
            return None
        main = torch.cuda.current_stream(self.device)
        fork = torch.cuda.Event()
        fork.record(main)
        # several frames in flight: binning kernels on the lanes' high-priority streams, render kernels on the library's
        # lowest-priority stream of each workspace (include/gs.h: gs_set_render_stream, set per workspace)
        host = None
        if to_host:
            if self._host_rgb is None or self._host_rgb.shape[0] < n:
                self._host_rgb = torch.empty((n, 3, self.H, self.W), dtype=torch.float32).pin_memory()
            host = self._host_rgb[:n]
            if self._copy_stream is None:
                self._copy_stream = torch.cuda.Stream(device=self.device)
        s = self.scene
        for i, cam in enumerate(cams):
            ln = self._lane(i % lanes)
            st = ln["stream"]
            if i < lanes:
                st.wait_event(fork)
            if ln["copy_pending"]:
                st.wait_event(ln["copied"])          # the image of frame i - lanes has left this lane's buffer
                ln["copy_pending"] = False
            img = ln["out_rgb"] if out_rgb is None else out_rgb[i]
            if ln["render_stream"] != (lanes > 1):     # a per-workspace switch: other renderers and threads are not affected
                binding.gs_set_workspace_option(ln["workspace"], binding.GS_OPT_RENDER_STREAM, 1 if lanes > 1 else 0)
                ln["render_stream"] = lanes > 1
            binding.gs_render(s["means3D"], s["scales"], s["rotations"], s["opacities"], s["sh"], s["sh_degree"],
                              cam.viewmatrix, cam.projmatrix, cam.fx, cam.fy, cam.W, cam.H, s["bg"], img,
                              ln["out_final_T"], ln["out_tile_counts"], None, ln["workspace"], st)
            ln["done"].record(st)
            if to_host:
                cs = self._copy_stream
                cs.wait_event(ln["done"])
                with torch.cuda.stream(cs):
                    host[i].copy_(img, non_blocking=True)
                ln["copied"].record(cs)
                ln["copy_pending"] = True
        for k in range(lanes):
            main.wait_event(self._lanes[k]["done"])
        if to_host:
            done = torch.cuda.Event()
            done.record(self._copy_stream)
            main.wait_event(done)
            for k in range(lanes):
                self._lanes[k]["copy_pending"] = False
        return host

    def close(self) -> None:
        """Releases what the library keeps for this renderer's workspaces (streams, events); the tensors go with the object."""
        wss = [self.workspace] + [ln["workspace"] for ln in (self._lanes or [])[1:]]
        for ws in wss:
            if ws is not None:
                binding.gs_release(ws)
        self._lanes = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def synchronize_readback(self) -> None:
        if self._ring is not None:
            self._ring["copy_stream"].synchronize()
        if self._copy_stream is not None:
            self._copy_stream.synchronize()
        torch.cuda.current_stream(self.device).synchronize()

    def read_image(self, slot: int = 0, n_slots: int = 1) -> torch.Tensor:
        """Async device -> pinned-host copy of the last frame's RGB image into host slot `slot`; returns the host
        tensor (valid after the stream is synchronised)."""
        if self._host_rgb is None or self._host_rgb.shape[0] < n_slots:
            self._host_rgb = torch.empty((n_slots, 3, self.H, self.W), dtype=torch.float32).pin_memory()
        self._host_rgb[slot].copy_(self.out_rgb, non_blocking=True)
        return self._host_rgb[slot]

    def intermediates(self, copy=("per_gaussian", "tile_ranges", "sorted_ids")):
        return binding.gs_get_intermediates(self.workspace, copy)
