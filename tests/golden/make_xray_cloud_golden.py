"""Writes tests/golden/xray_cloud.txt: three holes of the seeded X-ray cloud generator, computed WITHOUT oracle/.

    python tests/golden/make_xray_cloud_golden.py

Independent restatement in pure Python (arbitrary-precision integers for Philox4x32-10 of Salmon et al., SC'11, whose
published known-answer vectors pin the round function in tests/golden/philox_kat.txt; `math` for Box-Muller), of the
definition in DESIGN.md 6.7b: hole k = centre + sigma * n_k, n_k the Box-Muller triple of
Philox4x32-10(counter (k_lo, 'XRAY' = 0x58524159, k_hi, 0), key (gen_seed_lo, gen_seed_hi)) with the uniform mapping of
DESIGN.md R13, rounded to FP32 (a 3-D Gaussian initial cloud; FP32 state).  Imports nothing
from oracle/ or from the product."""
import math
import os
import struct

M0, M1, W0, W1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85
MASK = 0xFFFFFFFF


def philox4x32_10(ctr, key):
    c, k = list(ctr), list(key)
    for _ in range(10):
        p0, p1 = M0 * c[0], M1 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & MASK, (p0 >> 32) ^ c[3] ^ k[1], p0 & MASK]
        k = [(k[0] + W0) & MASK, (k[1] + W1) & MASK]
    return c


def f32(x):
    return struct.unpack("f", struct.pack("f", x))[0]


def hole(gen_seed, k, centre, sigma):
    w = philox4x32_10([k & MASK, 0x58524159, k >> 32, 0], [gen_seed & MASK, gen_seed >> 32])
    ua, fa = ((w[0] >> 9) + 0.5) / 2 ** 23, (w[1] >> 8) / 2 ** 24
    ub, fb = ((w[2] >> 9) + 0.5) / 2 ** 23, (w[3] >> 8) / 2 ** 24
    ra, rb = math.sqrt(-2.0 * math.log(ua)), math.sqrt(-2.0 * math.log(ub))
    return w, [f32(centre[0] + sigma * ra * math.cos(2.0 * math.pi * fa)),
               f32(centre[1] + sigma * ra * math.sin(2.0 * math.pi * fa)),
               f32(centre[2] + sigma * rb * math.cos(2.0 * math.pi * fb))]


if __name__ == "__main__":
    cases = [(0x1234567890ABCDEF, (1 << 32) + 9, (3.0, -7.0, 200.0), 0.8), (20220322, 0, (0.0, 0.0, 647.0), 0.05),
             (7, 131071, (-100.0, 250.0, 10.0), 2.0)]
    lines = ["# Three holes of the X-ray cloud generator, computed by tests/golden/make_xray_cloud_golden.py (pure Python,",
             "# no oracle code).  Definition: DESIGN.md 6.7b, R13; PAPER.md:100-102.",
             "# gen_seed index cx cy cz sigma | philox words w0..w3 (hex) | x y z (FP32, printed with 9 digits)"]
    for seed, k, c, s in cases:
        w, p = hole(seed, k, c, s)
        lines.append("%d %d %r %r %r %r %s %.9g %.9g %.9g" % (seed, k, c[0], c[1], c[2], s,
                                                          " ".join("%08x" % v for v in w), p[0], p[1], p[2]))
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "xray_cloud.txt")
    with open(out, "w") as f:
        f.write("\n".join(lines) + "\n")
    print(out)
