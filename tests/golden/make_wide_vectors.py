"""Re-derive tests/golden/wide_vectors.txt with plain big-integer arithmetic.

Independent of oracle/ and of the CUDA path: it restates readings A1, A4 and A19-A21 of DESIGN.md §3 (windows wider than
64 bits are folded to 64 bits before the hashes; the seed is masked to the window width, at most 64 bits) with Python
integers and prints the lines of the fixture.  Run:  python tests/golden/make_wide_vectors.py
"""
M64 = (1 << 64) - 1
GOLD = 0x9E3779B97F4A7C15


def fold64(hi, lo):
    t = (hi * GOLD) & M64
    return lo ^ (((t << 32) | (t >> 32)) & M64)


def g_bits(nbits, x):
    x ^= 0x5851F42D4C957F2D & ((1 << min(nbits, 64)) - 1)
    return (((x & 0xFFFFFFFF) ^ (x >> 32)) * 0x9E3779B1) & 0xFFFFFFFF


def f_bits(nbits, x):
    x ^= 0x2545F4914F6CDD1D & ((1 << min(nbits, 64)) - 1)
    h = ((x ^ (x >> 28)) * 0xD6E8FEB86659FD93) & M64
    return h ^ (h >> 32)


def window(v, total_bits, sym_bits, i, ln, k):
    """Sub(v, i, ln) of a k-symbol packed value, folded."""
    w = (v >> ((k - ln - i) * sym_bits)) & ((1 << (ln * sym_bits)) - 1)
    return fold64(w >> 64, w & M64)


if __name__ == "__main__":
    for hi, lo in ((0, 0), (0, 0x123456789ABCDEF0), (1, 0), (0xFFFFFFFFFFFFFFFF, 0), (0x0123456789ABCDEF, 0xFEDCBA9876543210),
                   ((1 << 56) - 1, 0x5555555555555555)):
        print("fold64 0x%X 0x%X = 0x%016X" % (hi, lo, fold64(hi, lo)))
    # g / f of folded windows of 62 (DNA m = 31), 120 (DNA s = 60), 125 (protein 25), 126 (triplet 21) and 30 bits (protein 6)
    for nbits, hi, lo in ((62, 0, (1 << 62) - 1), (120, (1 << 56) - 1, M64), (120, 0x00ABCDEF01234567, 0x89ABCDEF01234567),
                          (125, 0x1FFFFFFFFFFFFFFF, 0), (126, 0x2AAAAAAAAAAAAAAA, 0xAAAAAAAAAAAAAAAA), (30, 0, 0x2AAAAAAA)):
        x = fold64(hi, lo)
        print("g_bits %d 0x%X 0x%X = 0x%08X" % (nbits, hi, lo, g_bits(nbits, x)))
        print("f_bits %d 0x%X 0x%X = 0x%016X" % (nbits, hi, lo, f_bits(nbits, x)))
