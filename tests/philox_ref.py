"""Philox4x32-10 written a second time with Python big integers from the prose of DESIGN.md "C3"
(Salmon et al., SC'11).  Test-only; shares nothing with oracle/ or the CUDA path."""

M0 = 0xD2511F53
M1 = 0xCD9E8D57
W0 = 0x9E3779B9
W1 = 0xBB67AE85
MASK = 0xFFFFFFFF


def philox4x32_10(ctr, key):
    c = [int(x) & MASK for x in ctr]
    k = [int(x) & MASK for x in key]
    for r in range(10):
        p0 = M0 * c[0]
        p1 = M1 * c[2]
        c = [((p1 >> 32) ^ c[1] ^ k[0]) & MASK, p1 & MASK, ((p0 >> 32) ^ c[3] ^ k[1]) & MASK, p0 & MASK]
        k = [(k[0] + W0) & MASK, (k[1] + W1) & MASK]
    return c


def keyed(seed, c0, c1, c2, tag, step):
    return philox4x32_10([c0, c1, c2, (tag << 28) | step], [seed & MASK, (seed >> 32) & MASK])


def sweep_word(seed, step, slot, t, colour, q):
    """32-bit uniform of the active site with ordinal q in half-sweep (t, colour) of population slot `slot`
    (C3, reading G20): bit column p = q & 31 of the 32 keyed words of group q >> 5, word 0 = MSB"""
    gamma, p = q >> 5, q & 31
    u = 0
    for b in range(32):
        w = keyed(seed, slot, 8 * gamma + (b >> 2), 2 * t + colour, 2, step)[b & 3]
        u |= ((w >> p) & 1) << (31 - b)
    return u


def init_word(seed, j, v):
    return keyed(seed, v >> 2, j, 0, 0, 0)[v & 3]


def resample_uniform_fraction(seed, step, j, c):
    """exact rational numerator of u * 2^53: u = ((x>>12) + 0.5) * 2^-52  ->  (2*(x>>12) + 1) / 2^53"""
    w = keyed(seed, c >> 1, j, 0, 1, step)
    hi, lo = w[2 * (c & 1)], w[2 * (c & 1) + 1]
    x = (hi << 32) | lo
    return 2 * (x >> 12) + 1
