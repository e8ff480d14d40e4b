"""Derives the fp32 polynomial coefficients used in ul_math.cuh (run by hand; prints C literals).

Lawson-weighted least squares (converges to the minimax fit) in fp64, then the error of the
fp32 Horner evaluation is measured against numpy fp64 on a dense grid.  Nothing here is shared
with oracle/ (the oracle calls libm in fp64).
"""
import numpy as np


def lawson(basis, target, iters=200):
    w = np.ones(len(target))
    c = None
    for _ in range(iters):
        sw = np.sqrt(w)
        c, *_ = np.linalg.lstsq(basis * sw[:, None], target * sw, rcond=None)
        err = np.abs(basis @ c - target)
        w = w * (err + 1e-30)
        w /= w.sum()
    return c, np.abs(basis @ c - target).max()


def main():
    f32 = np.float32
    lim = np.pi / 4 + 0.01          # reduction may overshoot pi/4 slightly
    r = np.cos(np.linspace(0, np.pi, 20001)) * lim
    z = r * r
    # sin r = r + r z (S1 + S2 z + S3 z^2)
    c, e = lawson(np.stack([r * z, r * z * z, r * z ** 3], 1), np.sin(r) - r)
    print("sin", [repr(float(f32(v))) for v in c], "fit err %.3g" % e)
    S = [f32(v) for v in c]
    # cos r = 1 - z/2 + z^2 (C2 + C3 z + C4 z^2)
    c, e = lawson(np.stack([z * z, z ** 3, z ** 4], 1), np.cos(r) - 1 + z / 2)
    print("cos", [repr(float(f32(v))) for v in c], "fit err %.3g" % e)
    Cc = [f32(v) for v in c]
    rf = np.linspace(-lim, lim, 2000001).astype(f32)
    zf = rf * rf
    s = (S[2] * zf + S[1]) * zf + S[0]
    s = s * (zf * rf) + rf
    q = (Cc[2] * zf + Cc[1]) * zf + Cc[0]
    q = q * zf + f32(-0.5)
    q = q * zf + f32(1.0)
    print("fp32 eval max abs err: sin %.3g cos %.3g" % (np.abs(s.astype(np.float64) - np.sin(rf.astype(np.float64))).max(),
                                                         np.abs(q.astype(np.float64) - np.cos(rf.astype(np.float64))).max()))
    # atan q = q + q z (A1 + A2 z + A3 z^2 + A4 z^3 + A5 z^4) on |q| <= tan(pi/8) (+ slack)
    lim = np.tan(np.pi / 8) + 0.005
    x = np.cos(np.linspace(0, np.pi, 20001)) * lim
    z = x * x
    for n in (4, 5):
        c, e = lawson(np.stack([x * z ** (i + 1) for i in range(n)], 1), np.arctan(x) - x)
        print("atan", n, [repr(float(f32(v))) for v in c], "fit err %.3g" % e)
    A = [f32(v) for v in c]
    xf = np.linspace(-lim, lim, 2000001).astype(f32)
    zf = xf * xf
    p = A[4]
    for a in A[3::-1]:
        p = p * zf + a
    p = p * (zf * xf) + xf
    print("fp32 eval max abs err: atan %.3g" % np.abs(p.astype(np.float64) - np.arctan(xf.astype(np.float64))).max())


if __name__ == "__main__":
    main()
