"""Pins of oracle/projection.py (-m "not gpu"): what the mathematics fixes about a linear map followed by a rotary
embedding, chosen so that a dropped term, a wrong sign, a transposed weight or a wrong pairing fails one of them."""
import math

import numpy as np

from oracle import projection as P


def test_projection_is_the_plain_matrix_vector_product_loops():
    rng = np.random.default_rng(1)
    H, d, dm = 2, 4, 6
    Wq, Wk, Ww, h = rng.standard_normal((H * d, dm)), rng.standard_normal((H * d, dm)), rng.standard_normal((H, dm)), \
        rng.standard_normal(dm)
    q, k, w = P.project(h, Wq, Wk, Ww, pos=0, H_idx=H, d_idx=d, rope_dims=4, base=10000.0)
    for hd in range(H):
        for i in range(d):
            assert math.isclose(q[hd, i], sum(Wq[hd * d + i][j] * h[j] for j in range(dm)), rel_tol=1e-12, abs_tol=1e-12)
            assert math.isclose(k[hd, i], sum(Wk[hd * d + i][j] * h[j] for j in range(dm)), rel_tol=1e-12, abs_tol=1e-12)
        assert math.isclose(w[hd], sum(Ww[hd][j] * h[j] for j in range(dm)), rel_tol=1e-12, abs_tol=1e-12)


def test_rope_closed_forms():
    # base = 1: every pair turns by exactly `pos` radians
    x = np.zeros(8)
    x[1] = 1.0                                              # pair (1, 1 + 3) at rope_dims = 6
    y = P.rope_rotate(x, pos=0.5, rope_dims=6, base=1.0)
    assert math.isclose(y[1], math.cos(0.5)) and math.isclose(y[4], math.sin(0.5))
    assert np.count_nonzero(y) == 2
    x = np.zeros(8)
    x[4] = 1.0                                              # the partner: (-sin, cos)
    y = P.rope_rotate(x, pos=0.5, rope_dims=6, base=1.0)
    assert math.isclose(y[1], -math.sin(0.5)) and math.isclose(y[4], math.cos(0.5))
    # frequencies fall geometrically: angle[i] = pos * base^(-2i/rope)
    ang = P.rope_angles(3.0, 8, 10000.0)
    assert np.allclose(ang, [3.0, 3.0 * 10000 ** -0.25, 3.0 * 10000 ** -0.5, 3.0 * 10000 ** -0.75])
    # position 0 is the identity; dims beyond rope_dims never move
    z = np.random.default_rng(2).standard_normal((3, 10))
    assert np.array_equal(P.rope_rotate(z, 0, 6, 10000.0), z)
    assert np.array_equal(P.rope_rotate(z, 77, 6, 10000.0)[..., 6:], z[..., 6:])


def test_rope_is_a_rotation_and_depends_on_relative_position_only():
    rng = np.random.default_rng(3)
    x, y = rng.standard_normal(16), rng.standard_normal(16)
    for m, n, s in [(5, 2, 11), (100, 131071, 1000), (0, 7, 3)]:
        xm, yn = P.rope_rotate(x, m, 12, 1e6), P.rope_rotate(y, n, 12, 1e6)
        half = 6
        # every pair keeps its norm
        assert np.allclose(xm[:half] ** 2 + xm[half:12] ** 2, x[:half] ** 2 + x[half:12] ** 2)
        # <R_m x, R_n y> = <R_{m+s} x, R_{n+s} y>: the defining property of a rotary embedding
        a = xm @ yn
        b = P.rope_rotate(x, m + s, 12, 1e6) @ P.rope_rotate(y, n + s, 12, 1e6)
        assert math.isclose(a, b, rel_tol=1e-9, abs_tol=1e-9)
    # composition: rotating to m then by a further s (as positions add) equals rotating to m + s
    assert np.allclose(P.rope_rotate(P.rope_rotate(x, 4, 12, 1e6), 9, 12, 1e6), P.rope_rotate(x, 13, 12, 1e6))


def test_project_applies_rope_per_head_to_q_and_k_but_not_to_w():
    rng = np.random.default_rng(4)
    H, d, dm = 3, 8, 5
    Wq, Wk, Ww, h = rng.standard_normal((H * d, dm)), rng.standard_normal((H * d, dm)), rng.standard_normal((H, dm)), \
        rng.standard_normal(dm)
    q0, k0, w0 = P.project(h, Wq, Wk, Ww, 0, H, d, 4, 1e4)
    q9, k9, w9 = P.project(h, Wq, Wk, Ww, 9, H, d, 4, 1e4)
    assert np.array_equal(w0, w9)
    for hd in range(H):
        assert np.allclose(q9[hd], P.rope_rotate(q0[hd], 9, 4, 1e4)) and np.allclose(k9[hd], P.rope_rotate(k0[hd], 9, 4, 1e4))
    assert not np.allclose(q9[:, :4], q0[:, :4]) and np.array_equal(q9[:, 4:], q0[:, 4:])
