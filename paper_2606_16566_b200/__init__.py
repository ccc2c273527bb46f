"""B200-native forward 3D Gaussian Splatting tile rasterizer (Local-GS, arxiv/paper_2606_16566).

``binding`` is the ctypes layer over libgs.so (include/gs.h); ``renderer.Renderer`` is the small convenience object
that owns the output/workspace tensors of one camera size; ``scenes`` holds the seeded synthetic input generators.
Nothing in this package imports ``oracle`` (the CPU referee) and there is no CPU fallback.
"""
