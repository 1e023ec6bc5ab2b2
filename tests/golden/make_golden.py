"""Writes tests/golden/single_gaussian.txt from the closed form only (math/numpy; no oracle, no CUDA).

PAPER L78: G(x) = exp(-1/2 (x-mu)^T Sigma^-1 (x-mu)); L435: alpha = o G_2D(px), alpha_thresh = 1/255;
L86: c = sum c_i alpha_i T_i.  One isotropic Gaussian on the optical axis of a pinhole camera:
Sigma_2D = ((f s / z)^2 + 0.3) I (low-pass 0.3 = reading C4), alpha clamped at 0.99 (C11).
"""
import math
import os

F, Z, S, O = 80.0, 4.0, 0.25, 0.8
RGB = (0.2, 0.5, 0.9)
W = H = 64


def main():
    var = (F * S / Z) ** 2 + 0.3
    rows = ["# px py alpha r g b   (f=80 z=4 s=0.25 o=0.8 rgb=(0.2,0.5,0.9), 64x64, cx=cy=32)"]
    for py in range(0, H, 5):
        for px in range(0, W, 5):
            r2 = (px + 0.5 - 32.0) ** 2 + (py + 0.5 - 32.0) ** 2
            a = O * math.exp(-0.5 * r2 / var)
            a = min(0.99, a) if a >= 1.0 / 255.0 else 0.0
            rows.append("%d %d %.17g %.17g %.17g %.17g" % (px, py, a, a * RGB[0], a * RGB[1], a * RGB[2]))
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "single_gaussian.txt"), "w") as f:
        f.write("\n".join(rows) + "\n")


if __name__ == "__main__":
    main()
