"""Pins P3-P6, P10: Algorithms 3-7 (Eq. 2-3).

The literal bit-matrix oracle is compared with (a) numpy library routines
(unpackbits / roll / packbits), (b) a closed-form byte-level gather restated
here, (c) brute force over one-hot frames (bijectivity), (d) invariants.
"""
import numpy as np
import pytest


def np_reduction(F, D, B):
    """Eq. 2 / Eq. 3 via library routines: LSB-first bit rows rolled by d_h mod 8w,
    byte columns rolled by d_v mod h, XOR with B."""
    h, w, _ = F.shape
    out = np.empty_like(F)
    for c in range(3):
        bits = np.unpackbits(F[:, :, c], axis=1, bitorder="little")  # (h, 8w), column 8j+k = bit k
        for i in range(h):
            bits[i] = np.roll(bits[i], int(D[c * (h + w) + i]) % (8 * w))
        P = np.packbits(bits, axis=1, bitorder="little")
        for j in range(w):
            P[:, j] = np.roll(P[:, j], int(D[c * (h + w) + h + j]) % h)
        out[:, :, c] = P ^ B[:, :, c]
    return out


def closed_form(F, D, B):
    """F_e(ro,j,c) = B ^ ((F(i0,(j-q)%w,c) << r | F(i0,(j-q-1)%w,c) >> (8-r)) & 255),
    t = d_v(j,c) % h, i0 = (ro - t) % h, s = d_h(i0,c) % 8w, q = s >> 3, r = s & 7."""
    h, w, _ = F.shape
    out = np.empty_like(F)
    for c in range(3):
        for ro in range(h):
            for j in range(w):
                t = int(D[c * (h + w) + h + j]) % h
                i0 = (ro - t) % h
                s = int(D[c * (h + w) + i0]) % (8 * w)
                q, r = s >> 3, s & 7
                a = int(F[i0, (j - q) % w, c])
                b = int(F[i0, (j - q - 1) % w, c])
                out[ro, j, c] = (((a << r) | (b >> (8 - r))) & 0xFF) ^ int(B[ro, j, c])
    return out


def rnd(h, w, seed):
    rng = np.random.default_rng(seed)
    F = rng.integers(0, 256, (h, w, 3), dtype=np.uint8)
    D = rng.integers(0, 65536, 3 * (h + w), dtype=np.uint16)
    B = rng.integers(0, 256, (h, w, 3), dtype=np.uint8)
    return F, D, B


def test_bit_extract_is_unpackbits_little(orc):
    F, _, _ = rnd(5, 7, 0)
    M = orc.bit_extract(F)
    for c in range(3):
        assert (M[c] == np.unpackbits(F[:, :, c], axis=1, bitorder="little")).all()
    assert (orc.pack(M) == F).all()


def test_pack_is_lsb_first(orc):
    M = np.zeros((3, 1, 16), np.uint8)
    M[0, 0, 0] = 1   # bit 0 of pixel 0 -> value 1
    M[1, 0, 7] = 1   # bit 7 of pixel 0 -> value 128
    M[2, 0, 9] = 1   # bit 1 of pixel 1 -> value 2
    F = orc.pack(M)
    assert F[0, 0, 0] == 1 and F[0, 0, 1] == 128 and F[0, 1, 2] == 2 and F.sum() == 131


def test_hshift_vshift_are_rolls(orc):
    F, D, _ = rnd(6, 5, 1)
    h, w = 6, 5
    M = orc.bit_extract(F)
    Mh = orc.hshift(M, D)
    Mv = orc.vshift(M, D)
    for c in range(3):
        for i in range(h):
            assert (Mh[c, i] == np.roll(M[c, i], int(D[c * (h + w) + i]) % (8 * w))).all()
        for j in range(w):
            t = int(D[c * (h + w) + h + j]) % h
            assert (Mv[c][:, 8 * j:8 * j + 8] == np.roll(M[c][:, 8 * j:8 * j + 8], t, axis=0)).all()
    assert (orc.hshift(Mh, D, inverse=True) == M).all()
    assert (orc.vshift(Mv, D, inverse=True) == M).all()


def test_direction_is_scatter_towards_higher_index(orc):
    """Eq. 2 / Eq. 3 are written M[dest] = M[src] with dest = src + d: a set bit moves
    to a HIGHER bit column / row (reading Q12)."""
    h, w = 4, 4
    F = np.zeros((h, w, 3), np.uint8)
    F[1, 1, 0] = 0b00000100  # channel 0, row 1, bit column 8*1+2 = 10
    D = np.zeros(3 * (h + w), np.uint16)
    D[1] = 9          # d_h(row 1, c=0): bit column 10 -> 19 = pixel 2, bit 3
    D[h + 2] = 2      # d_v(column 2, c=0): row 1 -> 3
    E = orc.confuse_xor(F, D, np.zeros_like(F))
    want = np.zeros_like(F)
    want[3, 2, 0] = 0b00001000
    assert (E == want).all()


@pytest.mark.parametrize("h,w,seed", [(4, 4, 0), (7, 5, 1), (1, 9, 2), (9, 1, 3), (3, 16, 4), (16, 3, 5), (33, 20, 6)])
def test_literal_equals_numpy_and_closed_form(orc, h, w, seed):
    F, D, B = rnd(h, w, seed)
    E = orc.confuse_xor(F, D, B)
    assert (E == np_reduction(F, D, B)).all()
    assert (E == closed_form(F, D, B)).all()
    assert (orc.confuse_xor(E, D, B, inverse=True) == F).all()


def test_special_cases(orc):
    h, w = 6, 8
    F, D, B = rnd(h, w, 11)
    Z = np.zeros_like(B)
    D0 = np.zeros_like(D)
    assert (orc.confuse_xor(F, D0, Z) == F).all()                       # d = 0: identity
    assert (orc.confuse_xor(F, D0, B) == (F ^ B)).all()                 # XOR alone, B at the destination
    Dm = D0.copy()
    for c in range(3):
        Dm[c * (h + w): c * (h + w) + h] = 8 * w * 3                    # multiples of 8w: identity
        Dm[c * (h + w) + h: (c + 1) * (h + w)] = h * 5                  # multiples of h: identity
    assert (orc.confuse_xor(F, Dm, Z) == F).all()
    Db = D0.copy()
    Db[0:h] = 8 * 3                                                    # channel 0: pure byte roll by 3 pixels
    E = orc.confuse_xor(F, Db, Z)
    assert (E[:, :, 0] == np.roll(F[:, :, 0], 3, axis=1)).all()
    assert (E[:, :, 1:] == F[:, :, 1:]).all()


def test_brute_force_4x4_all_uniform_shifts(orc):
    """P5: every uniform (s, t) on a 4x4 frame: 32 bit shifts x 4 row shifts."""
    h = w = 4
    F, _, B = rnd(h, w, 21)
    for s in range(8 * w):
        for t in range(h):
            D = np.zeros(3 * (h + w), np.uint16)
            for c in range(3):
                D[c * (h + w): c * (h + w) + h] = s + 8 * w * c      # same residue, different raw value
                D[c * (h + w) + h: (c + 1) * (h + w)] = t + h * (c + 1)
            E = orc.confuse_xor(F, D, B)
            assert (E == closed_form(F, D, B)).all(), (s, t)


def test_brute_force_4x4_random_D(orc):
    h = w = 4
    rng = np.random.default_rng(22)
    F, _, B = rnd(h, w, 23)
    for it in range(2000):
        D = rng.integers(0, 65536, 3 * (h + w), dtype=np.uint16)
        E = orc.confuse_xor(F, D, B)
        assert (E == np_reduction(F, D, B)).all(), it
    # closed form on a subset (python loops)
    for it in range(200):
        D = rng.integers(0, 65536, 3 * (h + w), dtype=np.uint16)
        assert (orc.confuse_xor(F, D, B) == closed_form(F, D, B)).all()


@pytest.mark.parametrize("h,w", [(4, 4), (5, 3)])
def test_bijectivity_over_all_bit_positions(orc, h, w):
    """P4: the confusion is a permutation of the 24*w*h bit positions that never leaves the channel."""
    rng = np.random.default_rng(31)
    D = rng.integers(0, 65536, 3 * (h + w), dtype=np.uint16)
    Z = np.zeros((h, w, 3), np.uint8)
    nbits = 24 * w * h
    dest = np.empty(nbits, np.int64)
    for pos in range(nbits):
        byte, bit = divmod(pos, 8)
        F = np.zeros(3 * w * h, np.uint8)
        F[byte] = 1 << bit
        E = orc.confuse_xor(F.reshape(h, w, 3), D, Z).ravel()
        nz = np.flatnonzero(E)
        assert nz.size == 1 and bin(int(E[nz[0]])).count("1") == 1
        dest[pos] = nz[0] * 8 + int(E[nz[0]]).bit_length() - 1
        assert (nz[0] % 3) == (byte % 3)  # stays in its channel
    assert (np.sort(dest) == np.arange(nbits)).all()


def test_popcount_invariants(orc):
    """P6: with B = 0 the per-channel popcount is preserved; the horizontal step alone
    preserves per-row popcounts, the vertical step alone per-bit-column popcounts."""
    h, w = 12, 10
    F, D, _ = rnd(h, w, 41)
    E = orc.confuse_xor(F, D, np.zeros_like(F))
    for c in range(3):
        assert np.unpackbits(E[:, :, c]).sum() == np.unpackbits(F[:, :, c]).sum()
    M = orc.bit_extract(F)
    assert (orc.hshift(M, D).sum(axis=2) == M.sum(axis=2)).all()
    assert (orc.vshift(M, D).sum(axis=1) == M.sum(axis=1)).all()


def test_error_locality_no_diffusion(orc):
    """P10 (PAPER.md:647 and advantage (4)): corrupting one ciphertext byte changes at most two
    plaintext bytes, in the same channel, horizontally adjacent (mod w)."""
    h, w = 24, 20
    F, D, B = rnd(h, w, 51)
    E = orc.confuse_xor(F, D, B)
    rng = np.random.default_rng(52)
    for _ in range(20):
        i, j, c = int(rng.integers(h)), int(rng.integers(w)), int(rng.integers(3))
        E2 = E.copy()
        E2[i, j, c] ^= np.uint8(rng.integers(1, 256))
        P2 = orc.confuse_xor(E2, D, B, inverse=True)
        diff = np.argwhere(P2 != F)
        assert 1 <= len(diff) <= 2
        assert (diff[:, 2] == c).all()
        if len(diff) == 2:
            assert diff[0, 0] == diff[1, 0]
            assert (diff[1, 1] - diff[0, 1]) % w in (1, w - 1)
