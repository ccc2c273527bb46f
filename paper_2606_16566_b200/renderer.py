"""Renderer: owns the device copies of a scene, the output buffers and the workspace; one call = one frame.

This is the public Python API (the call a user makes).  It only allocates tensors and forwards to
binding.gs_render -- no arithmetic of the method lives here.
"""
from __future__ import annotations

import numpy as np
import torch

from . import binding


class Renderer:
    def __init__(self, P: int, W: int, H: int, max_dup: int, device="cuda:0", count_contrib: bool = True):
        self.P, self.W, self.H = int(P), int(W), int(H)
        self.device = torch.device(device)
        self.gx, self.gy = (W + 15) // 16, (H + 15) // 16
        self.max_dup = int(max_dup)
        nbytes = binding.gs_workspace_bytes(P, W, H, max_dup)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.out_rgb = torch.empty((3, H, W), dtype=torch.float32, device=self.device)
        self.out_final_T = torch.empty((H, W), dtype=torch.float32, device=self.device)
        self.out_tile_counts = torch.empty((self.gy * self.gx,), dtype=torch.int32, device=self.device)
        self.out_n_contrib = torch.empty((H, W), dtype=torch.int32, device=self.device) if count_contrib else None
        self.scene = None

    def upload(self, scene) -> None:
        """Host (numpy) scene -> device tensors (pinned staging, async copies on the current stream)."""
        def up(a):
            t = torch.from_numpy(np.ascontiguousarray(a))
            return t.pin_memory().to(self.device, non_blocking=True)
        self.scene = dict(means3D=up(scene.means3D), scales=up(scene.scales), rotations=up(scene.rotations),
                          opacities=up(scene.opacities), sh=up(scene.sh), sh_degree=int(scene.sh_degree),
                          bg=np.asarray(scene.bg, dtype=np.float32))

    def render(self, cam, stream=None) -> None:
        s = self.scene
        binding.gs_render(s["means3D"], s["scales"], s["rotations"], s["opacities"], s["sh"], s["sh_degree"],
                          cam.viewmatrix, cam.projmatrix, cam.fx, cam.fy, cam.W, cam.H, s["bg"], self.out_rgb,
                          self.out_final_T, self.out_tile_counts, self.out_n_contrib, self.workspace, stream)

    def intermediates(self, copy=("per_gaussian", "tile_ranges", "sorted_ids")):
        return binding.gs_get_intermediates(self.workspace, copy)
