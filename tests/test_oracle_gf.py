"""Pins for oracle step 6 (GF(2^128) multiply, SP 800-38D Algorithm 1).  SURVEY.md 8(c) pin table."""
import numpy as np

ONE = bytes([0x80]) + bytes(15)           # the polynomial "1": x^0 is the MSB of byte 0
X1 = bytes([0x40]) + bytes(15)            # the polynomial "x"
X127 = bytes(15) + bytes([0x01])          # x^127
R = bytes([0xE1]) + bytes(15)             # x^128 mod P = 1 + x + x^2 + x^7


def rnd(rng):
    return rng.integers(0, 256, 16, dtype=np.uint8).tobytes()


def xor(a, b):
    return bytes(p ^ q for p, q in zip(a, b))


def test_field_axioms(oracle):
    rng = np.random.default_rng(2001)
    for _ in range(300):
        a, b, c = rnd(rng), rnd(rng), rnd(rng)
        assert oracle.gf_mul(a, b) == oracle.gf_mul(b, a)
        assert oracle.gf_mul(oracle.gf_mul(a, b), c) == oracle.gf_mul(a, oracle.gf_mul(b, c))
        assert oracle.gf_mul(a, xor(b, c)) == xor(oracle.gf_mul(a, b), oracle.gf_mul(a, c))


def test_identity_and_zero(oracle):
    rng = np.random.default_rng(2002)
    for _ in range(50):
        a = rnd(rng)
        assert oracle.gf_mul(ONE, a) == a
        assert oracle.gf_mul(a, ONE) == a
        assert oracle.gf_mul(a, bytes(16)) == bytes(16)


def test_multiply_by_x_is_shift_with_conditional_reduce(oracle):
    rng = np.random.default_rng(2003)
    for _ in range(200):
        a = rnd(rng)
        v = int.from_bytes(a, "big")
        expect = v >> 1
        if v & 1:
            expect ^= 0xE1 << 120
        assert oracle.gf_mul(X1, a) == expect.to_bytes(16, "big")
    assert oracle.gf_mul(X1, X127) == R    # x * x^127 = x^128 = R


def test_frobenius_pins_the_reduction_polynomial(oracle):
    """Squaring is GF(2)-linear and a^(2^128) = a.  Both fail for a wrong reduction constant."""
    rng = np.random.default_rng(2004)
    for _ in range(10):
        a, b = rnd(rng), rnd(rng)
        sq = lambda t: oracle.gf_mul(t, t)
        assert sq(xor(a, b)) == xor(sq(a), sq(b))
        t = a
        for _ in range(128):
            t = sq(t)
        assert t == a


def test_pow_matches_repeated_multiplication(oracle):
    rng = np.random.default_rng(2005)
    h = rnd(rng)
    acc = ONE
    for e in range(0, 70):
        assert oracle.gf_pow(h, e) == acc
        acc = oracle.gf_mul(acc, h)
    # exponent laws on large exponents
    assert oracle.gf_mul(oracle.gf_pow(h, 123456789), oracle.gf_pow(h, 987654321)) == oracle.gf_pow(h, 1111111110)


# Second opinion: an independent formulation.  Bit-reflect the blocks into ordinary integers
# (coefficient of x^i at bit i), carry-less multiply as Python big integers, reduce modulo
# x^128 + x^7 + x^2 + x + 1, reflect back.
def _reflect(b):
    v = int.from_bytes(b, "big")
    return int(format(v, "0128b")[::-1], 2)


def _unreflect(v):
    return int(format(v, "0128b")[::-1], 2).to_bytes(16, "big")


def _clmul_mod(a, b):
    p = 0
    i = 0
    while b >> i:
        if (b >> i) & 1:
            p ^= a << i
        i += 1
    poly = (1 << 128) | 0x87
    for d in range(p.bit_length() - 1, 127, -1):
        if (p >> d) & 1:
            p ^= poly << (d - 128)
    return p


def test_second_opinion_bigint(oracle):
    rng = np.random.default_rng(2006)
    for _ in range(300):
        a, b = rnd(rng), rnd(rng)
        assert oracle.gf_mul(a, b) == _unreflect(_clmul_mod(_reflect(a), _reflect(b)))
