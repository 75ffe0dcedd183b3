#!/usr/bin/env python
"""Writes tests/golden/mask_vectors.txt: known-answer vectors of the stage-4 keep mask.

A restatement of DESIGN.md section 2.1 in Python big integers (every operation reduced mod 2^64
explicitly).  It imports NOTHING from this repository: the vectors pin the specification itself,
so a wrong constant or shift in either implementation (oracle/lya_oracle.c orc_keep, or the CUDA
keep_pair) fails against this file and says which side is wrong.

    python tests/golden/make_mask_vectors.py > tests/golden/mask_vectors.txt
"""
M = (1 << 64) - 1
GOLD = 0x9E3779B97F4A7C15
HI_XOR = 0xD1B54A32D192ED03
FIN = 0xD6E8FEB86659FD93


def mix64(z):
    z &= M
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M
    return z ^ (z >> 31)


def hash32(seed, a, b):
    lo, hi = min(a, b), max(a, b)
    klo = mix64(seed + lo * GOLD)
    khi = mix64((seed ^ HI_XOR) + hi * GOLD)
    x = (klo + khi) & M
    x ^= x >> 32
    x = (x * FIN) & M
    return x >> 32


def threshold(f):
    # floor(f * 2^32 + 0.5) clamped to [0, 2^32]; f is a decimal string so the value is exact here
    from fractions import Fraction
    t = int(Fraction(f) * (1 << 32) + Fraction(1, 2))
    return max(0, min(t, 1 << 32))


CASES = [  # (seed, a, b, reject fraction as text)
    (0, 0, 1, "0.5"), (0, 1, 0, "0.5"), (1, 0, 1, "0.5"), (2507001293, 12345, 67890, "0.99"),
    (2507001294, 52012515, 7, "0.99"), (2507001294, 7, 52012515, "0.99"), (0xFFFFFFFFFFFFFFFF, 3, 4, "0.9"),
    (42, 1 << 39, (1 << 39) + 1, "0.25"), (42, 5, 5000000000, "0.75"), (7, 100, 101, "0"), (7, 100, 101, "1"),
    (2507001290, 17, 1000, "0.97"), (11, 899999, 3, "0.9"), (12, 0, 2147483646, "0.5"),
]
# plus a scan that is guaranteed to contain kept and rejected pairs at f = 0.99
for k in range(400):
    CASES.append((2507001293, k, 100000 + 37 * k, "0.99"))
for k in range(200):
    CASES.append((2507001291, 3 * k + 1, 7 * k + 2000, "0.5"))

if __name__ == "__main__":
    print("# seed a b reject_fraction threshold hash32 keep   (DESIGN.md section 2.1; written by make_mask_vectors.py)")
    for seed, a, b, f in CASES:
        thr = threshold(f)
        h = hash32(seed, a, b)
        print(seed, a, b, f, thr, h, int(h >= thr))
