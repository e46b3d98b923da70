"""Writes the closed-form fixtures in this folder.  Uses only `math`; imports nothing from the
repo (neither oracle/ nor the CUDA package)."""
import math, os
here = os.path.dirname(os.path.abspath(__file__))

# periodic sinc row: N = Nd = 8, centre 4, theta = pi/5, delta at x=-2, y=1
nd, centre, th = 8, 4.0, math.pi / 5
t = -2 * math.cos(th) + 1 * math.sin(th)
row = []
for u in range(nd):
    tau = u - centre - t
    row.append(math.sin(math.pi * (nd - 1) * tau / nd) / (nd * math.sin(math.pi * tau / nd)))
with open(os.path.join(here, "dirichlet_delta_n8.txt"), "w") as fh:
    fh.write("# D(u - 4 - t), t = -2 cos(pi/5) + sin(pi/5); see README.md\n")
    fh.write(" ".join("%.13e" % v for v in row) + "\n")

# qGGMRF spot values, eq. (13): h = u^2/(c+u^(2-p)), h' = (1/sigma) u (2c + p u^(2-p))/(c+u^(2-p))^2
p, sigma, c = 1.2, 1 / 0.7, 1e-4
with open(os.path.join(here, "qggmrf_spot.txt"), "w") as fh:
    fh.write("# Delta h(Delta) h'(Delta)  for p=1.2 sigma=1/0.7 c=1e-4 (P:L159)\n")
    for D in (0.1, 1.0):
        u = D / sigma
        uq = u ** (2 - p)
        fh.write("%.1f %.13e %.13e\n" % (D, u * u / (c + uq), u * (2 * c + p * uq) / (c + uq) ** 2 / sigma))
