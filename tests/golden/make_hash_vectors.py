"""Re-derive tests/golden/hash_vectors.txt with plain big-integer arithmetic.

Independent of oracle/ and of the CUDA path: it restates readings A1, A2, A4, A5 of DESIGN.md §3
with Python integers and prints the lines of the fixture.  Run:  python tests/golden/make_hash_vectors.py
"""
M64 = (1 << 64) - 1


def g(m, x):
    x ^= 0x5851F42D4C957F2D & ((1 << (2 * m)) - 1)
    return (((x & 0xFFFFFFFF) ^ (x >> 32)) * 0x9E3779B1) & 0xFFFFFFFF


def sigma(key, P):
    return (((key * 0x9E3779B97F4A7C15) & M64) >> 32) >> (32 - P)


def f(s, x):
    x ^= 0x2545F4914F6CDD1D & ((1 << (2 * s)) - 1)
    h = ((x ^ (x >> 28)) * 0xD6E8FEB86659FD93) & M64
    return h ^ (h >> 32)


def bitpos(h, i, H):
    return (h >> (i * (64 // H))) & 63


if __name__ == "__main__":
    for m, x in ((16, 0), (16, 1), (16, 0xFFFFFFFF), (12, 0), (20, (1 << 40) - 1)):
        print("g %d 0x%X = 0x%08X" % (m, x, g(m, x)))
    for P in (12, 24, 0):
        print("sigma 0xB524331D %d = %d" % (P, sigma(0xB524331D, P)))
    for s, x in ((28, 0), (28, 1), (28, (1 << 56) - 1), (31, (1 << 62) - 1)):
        print("f %d 0x%X = 0x%016X" % (s, x, f(s, x)))
    h = f(28, 0)
    for i in range(4):
        print("bitpos 0x%016X %d 4 = %d" % (h, i, bitpos(h, i, 4)))
