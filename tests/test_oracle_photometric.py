"""Pins of oracle/photometric.py (masked photometric loss, Eq. 2; reading S20b) against things other
than itself: a library correlation routine, closed forms, symmetries and central finite differences."""
import numpy as np
import pytest
from scipy import ndimage

from oracle import photometric as ph


def rand_images(seed, H=23, W=31):
    rng = np.random.default_rng(seed)
    R = rng.uniform(0, 1, (3, H, W))
    I = np.clip(R + rng.normal(0, 0.1, (3, H, W)), 0, 1)
    M = (rng.uniform(0, 1, (H, W)) > 0.3).astype(np.uint8)
    return R, I, M


def test_window_is_normalised_separable_gaussian():
    G = ph.gaussian_window()
    assert G.shape == (11, 11) and abs(G.sum() - 1.0) < 1e-15
    assert np.allclose(G, G.T) and np.allclose(G, G[::-1, ::-1])
    assert np.linalg.matrix_rank(G) == 1
    # ratio of neighbouring taps along an axis: exp(-(1 - 0)/(2 sigma^2)) at the centre
    assert G[5, 6] / G[5, 5] == pytest.approx(np.exp(-1.0 / (2 * 1.5 ** 2)), rel=1e-14)


def test_window_sum_equals_library_correlation_with_zero_padding():
    rng = np.random.default_rng(0)
    a = rng.normal(size=(2, 19, 27))
    ref = np.stack([ndimage.correlate(a[c], ph.gaussian_window(), mode="constant", cval=0.0) for c in range(2)])
    assert np.abs(ph.window_sum(a) - ref).max() < 1e-14
    # a single impulse returns the (flipped = same) window
    imp = np.zeros((15, 15)); imp[7, 7] = 1.0
    assert np.allclose(ph.window_sum(imp)[2:13, 2:13], ph.gaussian_window())


def test_ssim_map_against_library_moments():
    R, I, _ = rand_images(1)
    G = ph.gaussian_window()
    S = ph.ssim_map(R, I)
    for c in range(3):
        f = lambda a: ndimage.correlate(a, G, mode="constant", cval=0.0)
        mx, my = f(R[c]), f(I[c])
        sxx, syy, sxy = f(R[c] ** 2) - mx ** 2, f(I[c] ** 2) - my ** 2, f(R[c] * I[c]) - mx * my
        ref = ((2 * mx * my + 1e-4) * (2 * sxy + 9e-4)) / ((mx ** 2 + my ** 2 + 1e-4) * (sxx + syy + 9e-4))
        assert np.abs(S[c] - ref).max() < 1e-12


def test_identical_images_have_ssim_one_zero_loss_zero_gradient():
    R, _, M = rand_images(2)
    out = ph.photometric_loss(R, R, M)
    assert np.abs(out["ssim_map"] - 1.0).max() < 1e-13
    assert out["loss"] == pytest.approx(0.0, abs=1e-14) and out["l1"] == 0.0
    assert np.abs(out["grad"]).max() < 1e-15


def test_constant_images_closed_form_in_the_interior():
    a, b = 0.7, 0.4
    x, y = np.full((3, 30, 30), a), np.full((3, 30, 30), b)
    S = ph.ssim_map(x, y)
    # interior pixels (window fully inside): mu = (a, b), variances 0  =>  SSIM = (2ab + C1)/(a^2 + b^2 + C1)
    assert np.abs(S[:, 5:25, 5:25] - (2 * a * b + 1e-4) / (a * a + b * b + 1e-4)).max() < 1e-11  # variances cancel to 1e-16 against C2 = 9e-4
    out = ph.photometric_loss(x, y, None, lam=0.0)
    assert out["loss"] == pytest.approx(abs(a - b), abs=1e-15)  # lam = 0: plain mean absolute error


def test_symmetry_and_mask_semantics():
    R, I, M = rand_images(3)
    assert np.abs(ph.ssim_map(R, I) - ph.ssim_map(I, R)).max() < 1e-14
    o1 = ph.photometric_loss(R, I, M)
    o2 = ph.photometric_loss(R * (M != 0), I * (M != 0), None)  # Eq. 2: L_c(I M, R M)
    assert o1["loss"] == pytest.approx(o2["loss"], abs=1e-15)
    # the render outside the mask cannot matter, and receives no gradient
    R2 = R.copy(); R2[:, M == 0] += 0.3
    assert ph.photometric_loss(R2, I, M)["loss"] == pytest.approx(o1["loss"], abs=1e-15)
    assert np.all(o1["grad"][:, M == 0] == 0.0)
    # all-background mask: both inputs vanish, SSIM = C1 C2 / (C1 C2) = 1, loss 0
    assert ph.photometric_loss(R, I, np.zeros_like(M))["loss"] == pytest.approx(0.0, abs=1e-15)


@pytest.mark.parametrize("lam", [0.2, 1.0])
def test_gradient_matches_central_finite_differences(lam):
    R, I, M = rand_images(4, H=17, W=20)
    out = ph.photometric_loss(R, I, M, lam=lam)
    g = out["grad"]
    rng = np.random.default_rng(5)
    h = 1e-6
    checked = 0
    for _ in range(40):
        c, yy, xx = rng.integers(0, 3), rng.integers(0, 17), rng.integers(0, 20)
        if abs(R[c, yy, xx] * (M[yy, xx] != 0) - I[c, yy, xx] * (M[yy, xx] != 0)) < 1e-4:
            continue  # |.| kink
        Rp, Rm = R.copy(), R.copy()
        Rp[c, yy, xx] += h; Rm[c, yy, xx] -= h
        fd = (ph.photometric_loss(Rp, I, M, lam=lam, want_grad=False)["loss"] -
              ph.photometric_loss(Rm, I, M, lam=lam, want_grad=False)["loss"]) / (2 * h)
        assert g[c, yy, xx] == pytest.approx(fd, rel=2e-5, abs=1e-10)
        checked += 1
    assert checked > 20
