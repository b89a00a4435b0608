"""Test-side, independently written Philox4x32-10 (pure Python ints) used to cross-check the
oracle's C routine and to brute-force tie-breaks (pin P9).  Salmon et al., SC'11."""
M0, M1 = 0xD2511F53, 0xCD9E8D57
W0, W1 = 0x9E3779B9, 0xBB67AE85
MASK = 0xFFFFFFFF


def philox4x32_10(ctr, key):
    c = [int(v) & MASK for v in ctr]
    k = [int(v) & MASK for v in key]
    for _ in range(10):
        p0 = M0 * c[0]
        p1 = M1 * c[2]
        c = [((p1 >> 32) ^ c[1] ^ k[0]) & MASK, p1 & MASK, ((p0 >> 32) ^ c[3] ^ k[1]) & MASK, p0 & MASK]
        k = [(k[0] + W0) & MASK, (k[1] + W1) & MASK]
    return c


def word0(seed, site, step, sim, purpose, aux=0):
    key = (seed & MASK, (seed >> 32) & MASK)
    return philox4x32_10((site, step, sim, purpose | (aux << 8)), key)[0]
