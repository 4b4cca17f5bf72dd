"""Regenerates the coefficients of atan2_pos() in lm_device.cuh: atan(t) = t + t^3 P(t^2) on [0, 1],
P of degree 7, iteratively re-weighted least squares (near-minimax); prints fp32 literals and the
achieved error.  Build-time helper of the CUDA path only (the oracle uses libm's atan2)."""
import numpy as np

N = 4000
x = np.cos(np.pi * (np.arange(N) + 0.5) / N) * 0.5 + 0.5
y = np.arctan(x) - x
A = np.stack([x ** (2 * k + 1) for k in range(1, 9)], 1)
w = np.ones(N)
for _ in range(300):
    c = np.linalg.lstsq(A * w[:, None], y * w, rcond=None)[0]
    e = np.abs(A @ c - y)
    w = w * (1 + e / e.max())
    w /= w.mean()
c32 = c.astype(np.float32)
print(", ".join("%.9ef" % v for v in c32))
t = np.linspace(0, 1, 400001).astype(np.float32)
t2 = t * t
p = np.full_like(t, c32[-1])
for k in range(len(c32) - 2, -1, -1):
    p = p * t2 + c32[k]
r = (p * t2 * t + t).astype(np.float64)
err = np.abs(r - np.arctan(t.astype(np.float64)))
print("fp32 abs err %.3e, rel err %.3e" % (err.max(), (err[1:] / np.arctan(t[1:].astype(np.float64))).max()))
