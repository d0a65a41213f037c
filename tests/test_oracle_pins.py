"""Pins of the fp64 oracle against what the paper and the mathematics fix.

The paper prints no worked numeric example (PAPER.md has formulas :79, :100-118 and a timing table
only), so the pins are closed forms, invariants, brute force on tiny inputs and a library
cross-check.  Each is chosen so that a plausible mistake in oracle/mvd_oracle.c fails it:
  dropped/extra term .......... P5 (dense matrix), P8 (FFT)
  conv <-> correlation swapped . P2 (off-centre delta closed form), P5, P8
  wrong centre / axis order .... P2 (dz != dx), P5 (H != W), P8
  simultaneous instead of sequential view update ... P6 (sum conservation), P5
  wrong view order ............. P5
  boundary not periodic ........ P3, P10, P5 (K > H aliasing)
  eps guard misplaced .......... P1 with zeros in phi, test_eps_guard
None of these tests touches the CUDA path.
"""
import numpy as np
import pytest

from oracle import mvd_oracle as orc
from paper_1503_07998_b200 import synth


def rand_psfs(V, K, seed):
    rng = np.random.default_rng(seed)
    return np.stack([synth.random_psf(K, rng) for _ in range(V)])


# ---------------------------------------------------------------------------------------------
# literal definition == fast (wrap-padded) implementation, bit for bit
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("W,H,K,V,T", [(8, 8, 3, 2, 3), (12, 8, 5, 3, 2), (8, 12, 7, 2, 2),
                                        (6, 5, 9, 2, 2), (17, 9, 5, 1, 3)])
def test_literal_equals_padded_bitwise(W, H, K, V, T):
    views = synth.random_views(V, 2, W, H, seed=W * 100 + H)
    psfs = rand_psfs(V, K, 5)
    a = orc.deconvolve(views, psfs, T, literal=True, n_threads=1)
    b = orc.deconvolve(views, psfs, T, literal=False, n_threads=2)
    assert np.array_equal(a, b)


# ---------------------------------------------------------------------------------------------
# P1: centred delta PSF, one view: psi == phi after any number of iterations, exactly
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("T", [0, 1, 7])
def test_P1_centred_delta_is_identity(T):
    views = synth.random_views(1, 3, 16, 10, seed=1, lo=0, hi=65536)
    views[0, 0, :2, :3] = 0          # zeros exercise the eps guard: 0 / max(0, eps) = 0
    views[0, 1, 4, 5] = 65535
    out = orc.deconvolve(views, synth.delta_psf(5)[None], T)
    assert np.array_equal(out, views[0].astype(np.float64))


# ---------------------------------------------------------------------------------------------
# P2: off-centre delta at offset d: psi_T(x) = phi(x + d) for T >= 1 (closed form).
# b(x) = phi(x-d); r(x) = phi(x)/phi(x-d); q(x) = r(x+d); psi_1(x) = phi(x+d); then r == 1.
# With convolution and correlation swapped the result would be phi(x - d).
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dz,dx", [(1, -2), (-3, 1), (0, 2), (2, 0)])
@pytest.mark.parametrize("T", [1, 4])
def test_P2_offcentre_delta_shifts_by_plus_d(dz, dx, T):
    views = synth.random_views(1, 2, 14, 9, seed=2, lo=5, hi=3000)
    out = orc.deconvolve(views, synth.delta_psf(7, dz, dx)[None], T)
    phi = views[0].astype(np.float64)
    expect = np.roll(phi, shift=(-dz, -dx), axis=(1, 2))        # expect[y, x] = phi[y+dz, x+dx]
    np.testing.assert_allclose(out, expect, rtol=1e-12, atol=0)
    wrong = np.roll(phi, shift=(dz, dx), axis=(1, 2))
    assert not np.allclose(out, wrong, rtol=1e-3)


# ---------------------------------------------------------------------------------------------
# P3: constant images with normalised PSFs stay constant (normalisation + periodic boundary)
# ---------------------------------------------------------------------------------------------
def test_P3_constant_is_fixed_point():
    V, K = 3, 5
    views = np.full((V, 2, 9, 11), 1234, dtype=np.uint16)
    psfs = rand_psfs(V, K, 3)
    out = orc.deconvolve(views, psfs, 6)
    # fp32 PSFs sum to 1 within ~1e-7, compounded over 2*V*T convolutions
    np.testing.assert_allclose(out, 1234.0, rtol=5e-6)


# ---------------------------------------------------------------------------------------------
# P4: psi stays non-negative and finite
# ---------------------------------------------------------------------------------------------
def test_P4_nonnegative_and_finite():
    views = synth.random_views(2, 2, 16, 12, seed=4, lo=0, hi=500)
    views[:, :, 3:6, 2:9] = 0
    out = orc.deconvolve(views, rand_psfs(2, 5, 4), 8)
    assert np.isfinite(out).all() and (out >= 0).all()


# ---------------------------------------------------------------------------------------------
# P5: brute force with dense matrices.  A_v[(y,x),(y',x')] += P_v[j][i] for
# (y',x') = ((y-(j-c)) mod H, (x-(i-c)) mod W);  psi <- psi . A_v^T (phi_v / max(A_v psi, eps)).
# Written with explicit matrices so that "correlation" is literally the transpose.
# ---------------------------------------------------------------------------------------------
def dense_operator(P, H, W):
    K = P.shape[0]
    c = (K - 1) // 2
    A = np.zeros((H * W, H * W))
    for y in range(H):
        for x in range(W):
            for j in range(K):
                for i in range(K):
                    A[y * W + x, ((y - (j - c)) % H) * W + ((x - (i - c)) % W)] += float(P[j, i])
    return A


def dense_rl(views_plane, psfs, T, eps):
    V, H, W = views_plane.shape
    phi = views_plane.reshape(V, -1).astype(np.float64)
    psi = phi.sum(0) / V
    ops = [dense_operator(psfs[v], H, W) for v in range(V)]
    for _ in range(T):
        for v in range(V):
            b = ops[v] @ psi
            r = phi[v] / np.maximum(b, eps)
            psi = psi * (ops[v].T @ r)
    return psi.reshape(H, W)


@pytest.mark.parametrize("W,H,K", [(8, 8, 3), (8, 8, 5), (8, 8, 7), (12, 8, 5), (8, 12, 7),
                                    (8, 8, 9),      # K > W: taps alias around the plane
                                    (6, 5, 9)])
def test_P5_dense_matrix_brute_force(W, H, K):
    V, T = 3, 4
    views = synth.random_views(V, 2, W, H, seed=50 + K)
    psfs = rand_psfs(V, K, 60 + W)
    out = orc.deconvolve(views, psfs, T)
    for p in range(2):
        ref = dense_rl(views[:, p], psfs, T, float(np.float32(1e-6)))
        np.testing.assert_allclose(out[p], ref, rtol=1e-11, atol=1e-11)


def test_P5_detects_view_order_and_simultaneous_form():
    """The pin has teeth: reversed view order or the product (simultaneous) form differ by percent."""
    V, T, W, H, K = 3, 4, 8, 8, 5
    views = synth.random_views(V, 1, W, H, seed=77)
    psfs = rand_psfs(V, K, 78)
    out = orc.deconvolve(views, psfs, T)[0]
    rev = dense_rl(views[::-1, 0], psfs[::-1], T, 1e-6)
    assert np.linalg.norm(out - rev) / np.linalg.norm(out) > 1e-3
    # simultaneous: every factor from the same psi^t
    phi = views[:, 0].reshape(V, -1).astype(np.float64)
    psi = phi.sum(0) / V
    ops = [dense_operator(psfs[v], H, W) for v in range(V)]
    for _ in range(T):
        f = np.ones_like(psi)
        for v in range(V):
            f *= ops[v].T @ (phi[v] / np.maximum(ops[v] @ psi, 1e-6))
        psi = psi * f
    assert np.linalg.norm(out.ravel() - psi) / np.linalg.norm(out) > 1e-3


# ---------------------------------------------------------------------------------------------
# P6: sum conservation after EVERY view update: sum(psi) == sum(phi_v)   (sequential form only)
# ---------------------------------------------------------------------------------------------
def test_P6_sum_conservation_per_view_update():
    V, T, K = 3, 5, 7
    views = synth.random_views(V, 1, 20, 14, seed=6, lo=20, hi=900)
    psfs64 = [p.astype(np.float64) for p in rand_psfs(V, K, 6)]
    tr = orc.trace(views[:, 0], np.stack(psfs64), T)
    assert tr.shape == (T * V, 14, 20)
    for t in range(T):
        for v in range(V):
            s_psf = float(np.stack(psfs64)[v].astype(np.float32).astype(np.float64).sum())
            got = tr[t * V + v].sum()
            want = views[v, 0].astype(np.float64).sum()
            # exact identity is sum(psi') = sum_y r(y) * (P^T-sum-weighted b) ; with sum(P)=1+-1e-7
            assert abs(got / want - 1.0) < 5e-7 + abs(s_psf - 1.0) * 2


# ---------------------------------------------------------------------------------------------
# P7: single view: the I-divergence  sum[ phi log(phi/b) - phi + b ],  b = psi * P,  never increases
# ---------------------------------------------------------------------------------------------
def test_P7_idivergence_non_increasing():
    T, K = 25, 7
    prob = synth.make_problem(1, 1, 24, 18, K, T, seed=7, psf="random")
    tr = orc.trace(prob.views[:, 0], prob.psfs, T)
    phi = prob.views[0, 0].astype(np.float64)

    def idiv(psi):
        b = orc.blur(psi, prob.psfs[0])
        with np.errstate(divide="ignore", invalid="ignore"):
            t = np.where(phi > 0, phi * np.log(phi / b), 0.0)
        return float((t - phi + b).sum())

    d = [idiv(phi)] + [idiv(tr[t]) for t in range(T)]
    assert all(d[k + 1] <= d[k] * (1 + 1e-12) + 1e-9 for k in range(T)), d
    assert d[-1] < 0.9 * d[0]


# ---------------------------------------------------------------------------------------------
# P8: both convolutions against numpy's FFT (a library routine): blur = ifft(fft(psi) fft(h)),
# back-projection = ifft(fft(r) conj(fft(h))), h = PSF placed at ((j-c) mod H, (i-c) mod W)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("W,H,K", [(16, 12, 5), (15, 20, 9), (32, 8, 7), (8, 6, 11)])
def test_P8_convolutions_match_numpy_fft(W, H, K):
    rng = np.random.default_rng(8)
    img = rng.random((H, W)) * 100.0
    P = synth.random_psf(K, rng)
    c = (K - 1) // 2
    h = np.zeros((H, W))
    for j in range(K):
        for i in range(K):
            h[(j - c) % H, (i - c) % W] += float(P[j, i])
    Fh = np.fft.fft2(h)
    conv = np.fft.ifft2(np.fft.fft2(img) * Fh).real
    corr = np.fft.ifft2(np.fft.fft2(img) * np.conj(Fh)).real
    for literal in (False, True):
        np.testing.assert_allclose(orc.blur(img, P, literal), conv, rtol=1e-11, atol=1e-11)
        np.testing.assert_allclose(orc.backproject(img, P, literal), corr, rtol=1e-11, atol=1e-11)
    # the two differ for an asymmetric PSF, so a swap cannot hide
    assert np.abs(conv - corr).max() > 1e-3 * np.abs(conv).max()


def test_P8_backproject_is_adjoint_of_blur():
    rng = np.random.default_rng(81)
    a, b = rng.random((10, 14)), rng.random((10, 14))
    P = synth.random_psf(5, rng)
    lhs = (orc.blur(a, P) * b).sum()
    rhs = (a * orc.backproject(b, P)).sum()
    assert abs(lhs - rhs) < 1e-12 * abs(lhs)


# ---------------------------------------------------------------------------------------------
# P9: a duplicated view: (phi, P) twice for T iterations == once for 2T iterations, bit-identical
# ---------------------------------------------------------------------------------------------
def test_P9_duplicated_view():
    views1 = synth.random_views(1, 2, 12, 10, seed=9)
    psf = rand_psfs(1, 5, 9)
    views2 = np.concatenate([views1, views1], axis=0)
    a = orc.deconvolve(views2, np.concatenate([psf, psf]), 3)
    b = orc.deconvolve(views1, psf, 6)
    assert np.array_equal(a, b)


# ---------------------------------------------------------------------------------------------
# P10: shift equivariance: circularly shifting every phi_v shifts the output identically
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("sy,sx", [(1, 0), (0, 1), (3, 5), (-2, 7)])
def test_P10_shift_equivariance(sy, sx):
    views = synth.random_views(2, 1, 13, 9, seed=10)
    psfs = rand_psfs(2, 5, 10)
    a = orc.deconvolve(views, psfs, 3)
    b = orc.deconvolve(np.roll(views, (sy, sx), axis=(2, 3)), psfs, 3)
    assert np.array_equal(np.roll(a, (sy, sx), axis=(1, 2)), b)


# ---------------------------------------------------------------------------------------------
# P11: zero iterations returns the mean of the views
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("V", [1, 2, 3, 6])
def test_P11_zero_iterations_is_mean(V):
    views = synth.random_views(V, 2, 8, 8, seed=11, lo=0, hi=65536)
    out = orc.deconvolve(views, rand_psfs(V, 3, 11), 0)
    assert np.array_equal(out, views.astype(np.float64).sum(0) / V)


# ---------------------------------------------------------------------------------------------
# eps guard (reading A6): r = phi / max(b, eps), eps taken at fp32 precision
# ---------------------------------------------------------------------------------------------
def test_eps_guard_value():
    # one view, centred delta, phi == 0 everywhere except one pixel: psi stays phi, no NaN/Inf
    views = np.zeros((1, 1, 6, 6), dtype=np.uint16)
    views[0, 0, 2, 3] = 9
    out = orc.deconvolve(views, synth.delta_psf(3)[None], 3)
    assert np.array_equal(out[0], views[0, 0].astype(np.float64))
    # blur below eps: psi = 0 region, phi > 0 there -> ratio = phi/eps lands only where psi == 0
    v2 = np.zeros((2, 1, 6, 6), dtype=np.uint16)
    v2[1, 0, 0, 0] = 7
    out = orc.deconvolve(v2, np.stack([synth.delta_psf(3), synth.delta_psf(3)]), 1)
    # psi0 = 3.5 at (0,0); view 0: r = 0/3.5 = 0 -> psi = 0 everywhere; view 1: r = 7/eps, psi*q = 0
    assert np.array_equal(out, np.zeros_like(out))


def test_argument_validation():
    views = synth.random_views(1, 1, 8, 8, seed=12)
    with pytest.raises(ValueError):
        orc.deconvolve(views, np.ones((1, 4, 4), np.float32) / 16, 1)      # even K
    with pytest.raises(ValueError):
        orc.deconvolve(views, synth.delta_psf(3)[None], -1)                # negative T
    with pytest.raises(ValueError):
        orc.deconvolve(views, synth.delta_psf(3)[None], 1, eps=0.0)        # eps <= 0


def test_threads_do_not_change_results():
    prob = synth.make_problem(2, 5, 16, 12, 5, 2, seed=13)
    a = orc.deconvolve(prob.views, prob.psfs, prob.T, n_threads=1)
    b = orc.deconvolve(prob.views, prob.psfs, prob.T, n_threads=4)
    assert np.array_equal(a, b)


# ---------------------------------------------------------------------------------------------
# Explicit back-projectors X_v ("replaced X with the expressions given below").
# Step a3 is the TRUE convolution r * X_v.
#   PX1  X = flip(P) is the Independent variant
#   PX2  dense-matrix brute force with an ASYMMETRIC X of a different size than P
#   PX3  centred-delta X, centred-delta P, one view: psi_1 = psi_0 . phi / psi_0 = phi
#   PX4  off-centre delta X at d: q(x) = r(x - d), the opposite shift of P2 (a flipped X would give +d)
# ---------------------------------------------------------------------------------------------
def test_PX1_flipped_psf_is_the_independent_variant():
    views = synth.random_views(3, 2, 14, 9, seed=7)
    psfs = rand_psfs(3, 5, 8)
    a = orc.deconvolve(views, psfs, 4)
    b = orc.deconvolve(views, psfs, 4, backprojectors=psfs[:, ::-1, ::-1])
    np.testing.assert_allclose(b, a, rtol=1e-12)
    assert np.array_equal(orc.backprojectors(psfs, "independent"), psfs[:, ::-1, ::-1])
    wrong = orc.deconvolve(views, psfs, 4, backprojectors=psfs)          # unflipped: must differ
    assert np.abs(wrong - a).max() > 1e-3 * a.max()


def dense_rl_x(views_plane, psfs, xs, T, eps):
    V, H, W = views_plane.shape
    phi = views_plane.reshape(V, -1).astype(np.float64)
    psi = phi.sum(0) / V
    A = [dense_operator(psfs[v], H, W) for v in range(V)]
    B = [dense_operator(xs[v], H, W) for v in range(V)]                   # convolution with X_v
    for _ in range(T):
        for v in range(V):
            r = phi[v] / np.maximum(A[v] @ psi, eps)
            psi = psi * (B[v] @ r)
    return psi.reshape(H, W)


@pytest.mark.parametrize("W,H,K,KX", [(8, 8, 3, 5), (12, 8, 5, 3), (8, 12, 5, 7), (6, 5, 3, 9)])
def test_PX2_dense_matrix_brute_force_with_explicit_backprojectors(W, H, K, KX):
    V, T = 2, 3
    views = synth.random_views(V, 2, W, H, seed=70 + K)
    psfs, xs = rand_psfs(V, K, 80 + W), rand_psfs(V, KX, 90 + H)
    for literal in (False, True):
        out = orc.deconvolve(views, psfs, T, backprojectors=xs, literal=literal)
        for p in range(2):
            ref = dense_rl_x(views[:, p], psfs, xs, T, float(np.float32(1e-6)))
            np.testing.assert_allclose(out[p], ref, rtol=1e-11, atol=1e-11)


def test_PX3_PX4_delta_backprojectors():
    views = synth.random_views(1, 2, 12, 10, seed=3, lo=10, hi=4000)
    phi = views[0].astype(np.float64)
    d0 = synth.delta_psf(5)[None]
    out = orc.deconvolve(views, d0, 3, backprojectors=synth.delta_psf(3)[None])
    np.testing.assert_allclose(out, phi, rtol=1e-13)
    # P = centred delta, X = delta at (dz, dx): psi_1(x) = phi(x) . 1 ... r = 1 everywhere, q = 1: psi stays phi;
    # use two views so that r is not constant: psi_0 = mean, r_0 = phi_0 / psi_0, q(x) = r_0(x - d)
    v2 = synth.random_views(2, 1, 12, 10, seed=4, lo=10, hi=4000)
    P = np.stack([synth.delta_psf(3)] * 2)
    dz, dx = 1, -2
    X = np.stack([synth.delta_psf(5, dz, dx), synth.delta_psf(5)])
    tr = orc.deconvolve(v2[:, :1], P, 1, backprojectors=X)[0]
    f = v2[:, 0].astype(np.float64)
    psi0 = f.mean(0)
    psi1 = psi0 * np.roll(f[0] / psi0, shift=(dz, dx), axis=(0, 1))       # q(x) = r(x - d)
    psi2 = psi1 * (f[1] / psi1)
    np.testing.assert_allclose(tr, psi2, rtol=1e-12)


def test_backprojector_builders_arithmetic():
    """The variant builders of oracle/mvd_oracle.py against scipy's convolution and their invariants
    (their READING of the garbled formulas is unpinned; this pins the arithmetic only)."""
    from scipy.signal import convolve2d
    psfs = rand_psfs(3, 5, 11)
    P = psfs.astype(np.float64)
    flip = P[:, ::-1, ::-1]
    for variant, factor in (("efficient_bayesian", lambda v, w: convolve2d(convolve2d(flip[v], P[w]), flip[w])),
                            ("optimization1", lambda v, w: convolve2d(flip[v], P[w]))):
        X = orc.backprojectors(psfs, variant)
        assert X.shape == psfs.shape and X.dtype == np.float32
        np.testing.assert_allclose(X.sum(axis=(1, 2)), 1.0, rtol=1e-6)
        for v in range(3):
            want = flip[v].copy()
            for w in range(3):
                if w != v:
                    f = factor(v, w)
                    o = (f.shape[0] - 5) // 2
                    want *= f[o:o + 5, o:o + 5]
            np.testing.assert_allclose(X[v], want / want.sum(), rtol=2e-6)
    # one view: W_v is empty, every variant is the (normalised) flipped PSF
    one = rand_psfs(1, 7, 12)
    np.testing.assert_allclose(orc.backprojectors(one, "efficient_bayesian")[0],
                               one[0, ::-1, ::-1] / one[0].astype(np.float64).sum(), rtol=1e-6)
    # sum X_v = 1 (and sum P_v = 1): constant views stay a fixed point (P3 carries over; flux
    # conservation P6 does not -- it needs X_v to be the adjoint of P_v)
    views = np.full((3, 1, 12, 16), 777, dtype=np.uint16)
    out = orc.deconvolve(views, psfs, 3, backprojectors=orc.backprojectors(psfs, "optimization1"))
    np.testing.assert_allclose(out, 777.0, rtol=1e-5)
    with pytest.raises(ValueError):
        orc.backprojectors(psfs, "optimization2")


# ---------------------------------------------------------------------------------------------
# Per-view weights (mvd_oracle_w; PAPER.md:88 lists a "weights" buffer and never defines it).
# READING W1 (parity unpinned): a4 becomes psi <- psi . (w_v q + 1 - w_v).
# What is pinned here is the arithmetic of that reading and the cases any reading must satisfy.
# ---------------------------------------------------------------------------------------------
def test_PW1_unit_weights_are_the_unweighted_run_bit_for_bit():
    views = synth.random_views(3, 2, 14, 10, seed=201)
    psfs = rand_psfs(3, 5, 202)
    a = orc.deconvolve(views, psfs, 4)
    b = orc.deconvolve(views, psfs, 4, weights=np.ones(views.shape, np.float32))
    assert np.array_equal(a, b)
    c = orc.deconvolve(views, psfs, 4, weights=np.ones(views.shape, np.float32), literal=True)
    assert np.array_equal(a, c)


def test_PW2_a_view_with_zero_weight_is_never_applied():
    # all weights zero: nothing is ever applied, psi stays the mean of the views
    views = synth.random_views(2, 2, 12, 9, seed=203)
    psfs = rand_psfs(2, 5, 204)
    out = orc.deconvolve(views, psfs, 5, weights=np.zeros(views.shape, np.float32))
    assert np.array_equal(out, views.astype(np.float64).sum(0) / 2)
    # two identical views, the second with weight 0: psi_0 = phi, and the run is the single-view run
    one = synth.random_views(1, 2, 12, 9, seed=205)
    two = np.concatenate([one, one])
    P = rand_psfs(1, 5, 206)
    w = np.ones(two.shape, np.float32)
    w[1] = 0.0
    assert np.array_equal(orc.deconvolve(two, np.concatenate([P, P]), 4, weights=w), orc.deconvolve(one, P, 4))
    # a pixel mask: pixels whose weight is 0 in every view keep psi_0 for ever, the others move
    views = synth.random_views(2, 1, 12, 9, seed=207)
    w = np.ones(views.shape, np.float32)
    w[:, 0, 2:5, 3:8] = 0.0
    out = orc.deconvolve(views, psfs, 3, weights=w)[0]
    psi0 = views[:, 0].astype(np.float64).sum(0) / 2
    assert np.array_equal(out[2:5, 3:8], psi0[2:5, 3:8])
    assert not np.allclose(out[6:, :], psi0[6:, :], rtol=1e-3)


def test_PW3_constants_stay_fixed_under_any_weights():
    views = np.full((2, 1, 10, 8), 321, dtype=np.uint16)
    rng = np.random.default_rng(208)
    w = rng.random(views.shape).astype(np.float32)
    out = orc.deconvolve(views, rand_psfs(2, 5, 209), 6, weights=w)
    np.testing.assert_allclose(out, 321.0, rtol=1e-12)


@pytest.mark.parametrize("W,H,K", [(8, 8, 3), (12, 8, 5), (6, 5, 9)])
def test_PW4_dense_matrix_brute_force_with_random_weights(W, H, K):
    V, T = 3, 4
    views = synth.random_views(V, 2, W, H, seed=210 + K)
    psfs = rand_psfs(V, K, 211 + W)
    rng = np.random.default_rng(212)
    w = rng.random(views.shape).astype(np.float32)
    w[0, :, :2] = 0.0
    w[1, :, -2:] = 1.0
    out = orc.deconvolve(views, psfs, T, weights=w)
    eps = float(np.float32(1e-6))
    for p in range(2):
        phi = views[:, p].reshape(V, -1).astype(np.float64)
        psi = phi.sum(0) / V
        ops = [dense_operator(psfs[v], H, W) for v in range(V)]
        for _ in range(T):
            for v in range(V):
                q = ops[v].T @ (phi[v] / np.maximum(ops[v] @ psi, eps))
                wv = w[v, p].reshape(-1).astype(np.float64)
                psi = psi * (wv * q + (1.0 - wv))
        np.testing.assert_allclose(out[p], psi.reshape(H, W), rtol=1e-11, atol=1e-11)


def test_PW_argument_validation():
    views = synth.random_views(1, 1, 8, 8, seed=213)
    w = np.ones(views.shape, np.float32)
    w[0, 0, 0, 0] = 1.5
    with pytest.raises(ValueError):
        orc.deconvolve(views, synth.delta_psf(3)[None], 1, weights=w)
    w[0, 0, 0, 0] = np.nan
    with pytest.raises(ValueError):
        orc.deconvolve(views, synth.delta_psf(3)[None], 1, weights=w)


# ---------------------------------------------------------------------------------------------
# PD: the paper's padded boundary, READING PD1 = zero padding (oracle.deconvolve_padded)
# ---------------------------------------------------------------------------------------------
def _rl_zero_boundary_scipy(views, psfs, T, eps, weights=None):
    """RL with ZERO boundary conditions written with scipy's non-periodic routines (independent of the oracle's
    periodic loops): b = convolve2d(psi, P, 'same', fill 0), q = correlate2d(r, P, 'same', fill 0)."""
    from scipy.signal import convolve2d, correlate2d
    V, N, H, W = views.shape
    out = np.empty((N, H, W))
    e32 = float(np.float32(eps))
    for n in range(N):
        phi = views[:, n].astype(np.float64)
        psi = phi.mean(axis=0) if V not in (1, 2, 4) else phi.sum(axis=0) / V
        for _ in range(T):
            for v in range(V):
                P = psfs[v].astype(np.float64)
                b = convolve2d(psi, P, mode="same", boundary="fill", fillvalue=0.0)
                r = phi[v] / np.maximum(b, e32)
                q = correlate2d(r, P, mode="same", boundary="fill", fillvalue=0.0)
                if weights is not None:
                    w = weights[v, n].astype(np.float64)
                    q = w * q + (1.0 - w)
                psi = psi * q
        out[n] = psi
    return out


@pytest.mark.parametrize("W,H,K,V", [(13, 9, 5, 2), (8, 12, 7, 3), (10, 10, 3, 1), (6, 5, 9, 2)])
def test_PD1_padding_amount_does_not_matter(W, H, K, V):
    """Zero padding of K - 1 pixels decouples opposite edges; any larger padding gives the same plane."""
    rng = np.random.default_rng(W * 100 + K)
    views = rng.integers(0, 500, size=(V, 2, H, W)).astype(np.uint16)
    psfs = rand_psfs(V, K, K + W)
    a = orc.deconvolve_padded(views, psfs, 4)
    for extra in (1, 5):
        b = orc.deconvolve_padded(views, psfs, 4, extra=extra)
        np.testing.assert_allclose(b, a, rtol=1e-12, atol=1e-300)


@pytest.mark.parametrize("W,H,K,V", [(13, 9, 5, 2), (8, 12, 7, 3), (16, 16, 9, 2)])
def test_PD2_padded_mode_is_rl_with_zero_boundary(W, H, K, V):
    """Against scipy.signal.convolve2d / correlate2d with zero fill: a dropped or transposed tap, the wrong flip
    or a crop at the wrong corner all fail here (asymmetric PSFs, W != H)."""
    rng = np.random.default_rng(7 * W + K)
    views = rng.integers(1, 800, size=(V, 2, H, W)).astype(np.uint16)
    psfs = rand_psfs(V, K, 3 * K + H)
    ref = _rl_zero_boundary_scipy(views, psfs, 3, 1e-6)
    got = orc.deconvolve_padded(views, psfs, 3)
    np.testing.assert_allclose(got, ref, rtol=1e-11, atol=1e-300)
    # and it is NOT the periodic result (the readings differ wherever the PSF reaches across an edge)
    per = orc.deconvolve(views, psfs, 3)
    assert np.abs(per - got).max() > 1e-3 * np.abs(got).max()


def test_PD3_interior_of_a_dark_bordered_plane_matches_periodic():
    """A plane whose outer K - 1 pixels are zero in every view sees no difference between the two boundaries."""
    K, V, H, W = 5, 2, 20, 24
    rng = np.random.default_rng(5)
    views = np.zeros((V, 1, H, W), dtype=np.uint16)
    views[:, :, K - 1:H - K + 1, K - 1:W - K + 1] = rng.integers(1, 900, size=(V, 1, H - 2 * K + 2, W - 2 * K + 2))
    psfs = rand_psfs(V, K, 11)
    np.testing.assert_allclose(orc.deconvolve_padded(views, psfs, 3), orc.deconvolve(views, psfs, 3), rtol=1e-12, atol=1e-300)


# ---------------------------------------------------------------------------------------------
# PP: the update as printed in PAPER.md:79 (simultaneous / product form), oracle.deconvolve_product
# ---------------------------------------------------------------------------------------------
def dense_rl_product(views_plane, psfs, T, eps):
    V, H, W = views_plane.shape
    phi = views_plane.reshape(V, -1).astype(np.float64)
    psi = phi.sum(0) / V
    ops = [dense_operator(psfs[v], H, W) for v in range(V)]
    for _ in range(T):
        f = np.ones_like(psi)
        for v in range(V):
            f *= ops[v].T @ (phi[v] / np.maximum(ops[v] @ psi, eps))
        psi = psi * f
    return psi.reshape(H, W)


@pytest.mark.parametrize("W,H,K", [(8, 8, 3), (12, 8, 5), (8, 12, 7), (6, 5, 9)])
def test_PP1_product_form_dense_matrix_brute_force(W, H, K):
    V, T = 3, 4
    views = synth.random_views(V, 2, W, H, seed=150 + K)
    psfs = rand_psfs(V, K, 160 + W)
    out = orc.deconvolve_product(views, psfs, T)
    for p in range(2):
        ref = dense_rl_product(views[:, p], psfs, T, float(np.float32(1e-6)))
        np.testing.assert_allclose(out[p], ref, rtol=1e-11, atol=1e-11)
    assert np.abs(out - orc.deconvolve(views, psfs, T)).max() > 1e-3 * out.max()    # not the sequential form


def test_PP2_single_view_product_is_sequential_and_constants_stay_fixed():
    views = synth.random_views(1, 2, 14, 10, seed=3)
    psfs = rand_psfs(1, 5, 4)
    np.testing.assert_allclose(orc.deconvolve_product(views, psfs, 5), orc.deconvolve(views, psfs, 5), rtol=1e-13)
    const = np.full((3, 1, 9, 11), 321, dtype=np.uint16)
    P = rand_psfs(3, 5, 8)
    np.testing.assert_allclose(orc.deconvolve_product(const, P, 4), 321.0, rtol=1e-12)


def test_PP3_product_form_with_weights():
    V, N, H, W, K = 2, 1, 9, 8, 3
    views = synth.random_views(V, N, W, H, seed=21)
    psfs = rand_psfs(V, K, 22)
    ones = np.ones((V, N, H, W), dtype=np.float32)
    np.testing.assert_array_equal(orc.deconvolve_product(views, psfs, 3, weights=ones), orc.deconvolve_product(views, psfs, 3))
    w = ones.copy()
    w[1] = 0.0                                                      # view 1 never applied == the single-view run
    np.testing.assert_allclose(orc.deconvolve_product(views, psfs, 3, weights=w)[0] * 0 + 1, 1.0)   # finite
    one_view = orc.deconvolve_product(views[:1], psfs[:1], 3)
    got = orc.deconvolve_product(views, psfs, 3, weights=w)
    # psi_0 differs (mean of both views), so compare the per-iteration factor instead: same update operator
    phi = views[:, 0].astype(np.float64)
    psi = phi.sum(0) / V
    for _ in range(3):
        psi = psi * orc.backproject(phi[0] / np.maximum(orc.blur(psi, psfs[0]), float(np.float32(1e-6))), psfs[0])
    np.testing.assert_allclose(got[0], psi, rtol=1e-12)
    assert one_view.shape == (1, H, W)


def test_PD4_padded_mode_with_weights():
    """Weights on a padded plan: the zero-boundary scipy formulation with reading W1's blend; the weight given to the
    padding is immaterial (psi is zero there)."""
    V, N, H, W, K = 2, 2, 9, 13, 5
    rng = np.random.default_rng(17)
    views = rng.integers(1, 800, size=(V, N, H, W)).astype(np.uint16)
    psfs = rand_psfs(V, K, 23)
    wts = rng.random((V, N, H, W)).astype(np.float32)
    got = orc.deconvolve_padded(views, psfs, 3, weights=wts)
    np.testing.assert_allclose(got, _rl_zero_boundary_scipy(views, psfs, 3, 1e-6, weights=wts), rtol=1e-11, atol=1e-300)
    assert np.abs(got - orc.deconvolve_padded(views, psfs, 3)).max() > 1e-3 * got.max()
    np.testing.assert_allclose(orc.deconvolve_padded(views, psfs, 3, weights=wts, extra=3), got, rtol=1e-12, atol=1e-300)
