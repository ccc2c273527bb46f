"""Writes tests/golden/t1_closed_form.txt from the CLOSED FORM only (no oracle, no CUDA code).

Pin T1 (BASELINE.json north_star (a)): one isotropic Gaussian of scale s on the optical axis at
depth z0, degree-0 colour c, opacity o, renders at distance r from its centre as
    rgb = bg*(1-alpha) + c*alpha,   alpha = o*exp(-r^2 / (2 sigma'^2)),   sigma'^2 = (f*s/z0)^2 + 0.3,
with alpha -> 0 below 1/255 and the 3-sigma rect of PAPER.md:53.  Run: python tests/golden/make_t1_closed_form.py
"""
import math
import os

W = H = 33
f, z0, s, o = 40.0, 4.0, 0.1, 0.7
c = (0.9, 0.5, 0.1)
bg = (0.2, 0.3, 0.4)
sig2 = (f * s / z0) ** 2 + 0.3
mu = ((W - 1) / 2.0, (H - 1) / 2.0)
lam = sig2 + math.sqrt(0.1)          # larger eigenvalue with the discriminant floored at 0.1 (reading S5)
radius = math.ceil(3.0 * math.sqrt(lam))
lines = ["# T1 closed-form fixture; see make_t1_closed_form.py (closed form of BASELINE.json north_star (a))",
         "# W H f z0 s o cr cg cb bgr bgg bgb",
         "params %d %d %r %r %r %r %r %r %r %r %r %r" % ((W, H, f, z0, s, o) + c + bg),
         "# sigma2 radius mu_x mu_y", "derived %.17g %d %.17g %.17g" % (sig2, radius, mu[0], mu[1]),
         "# x y alpha r g b T"]
for (x, y) in [(16, 16), (17, 16), (17, 17), (18, 16), (19, 17), (20, 16), (19, 19), (12, 16), (16, 13), (0, 0), (32, 32)]:
    r2 = (x - mu[0]) ** 2 + (y - mu[1]) ** 2
    a = min(0.99, o * math.exp(-r2 / (2.0 * sig2)))
    if a < 1.0 / 255.0:
        a = 0.0
    # the 3-sigma square rect in tiles truncates the splat (reading S6 / T4): tiles [0,2)x[0,2) of the 3x3 grid
    x0 = math.floor((mu[0] - radius) / 16.0); x1 = math.floor((mu[0] + radius + 15.0) / 16.0)
    if not (x0 <= x // 16 < x1 and x0 <= y // 16 < x1):
        a = 0.0
    rgb = [bg[k] * (1.0 - a) + c[k] * a for k in range(3)]
    lines.append("pixel %d %d %.12f %.12f %.12f %.12f %.12f" % (x, y, a, rgb[0], rgb[1], rgb[2], 1.0 - a))
open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "t1_closed_form.txt"), "w").write("\n".join(lines) + "\n")
