"""The one piece of arithmetic the paper prints next to the path: the 96-bit nonce collision bound.
It fixes the nonce length the container uses (12 bytes = 96 bits, reading S5 / F5): with any other length the printed
probabilities do not come out."""
import os

import workloads

HERE = os.path.dirname(os.path.abspath(__file__))


def test_nonce_collision_bound_matches_the_paper():
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "nonce_collision.txt")) if not l.startswith("#")]
    assert len(rows) == 2
    f = workloads.fits_frame(seed=1, ny=2, nx=2, n_sources=0)
    nonce_bits = 8 * len(f.nonce_d)
    assert nonce_bits == 96 and len(f.nonce_h) == 12
    for n_txt, p_txt in rows:
        n, printed = float(n_txt), float(p_txt)
        p = n * n / (2.0 * 2.0 ** nonce_bits)
        assert abs(p - printed) / printed < 0.01, (n, p, printed)      # the paper prints two significant digits
        wrong = n * n / (2.0 * 2.0 ** 128)                              # a 128-bit nonce would not reproduce it
        assert abs(wrong - printed) / printed > 0.5
