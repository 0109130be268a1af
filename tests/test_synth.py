"""Host-side checks of the seeded input generator (no GPU, no oracle arithmetic)."""
import numpy as np

from paper_1505_07674_b200 import synth


def test_configs_have_the_baseline_shapes():
    want = [(32, 32, 9, 4, None, 16), (100, 100, 22, 9, (9, 9), 1024), (200, 200, 29, 16, (21, 21), 4096),
            (256, 256, 43, 25, (15, 15), 4096), (512, 512, 22, 16, (31, 31), 16384),
            (120, 120, 19, 49, (15, 15), 4096)]                 # 5 = the paper's mock scenario (context)
    for c, (H, W, P, N, psf, B) in enumerate(want):
        cfg = synth.get_config(c)
        assert (cfg.H, cfg.W, cfg.P, len(cfg.quad), cfg.B) == (H, W, P, N, B)
        assert (None if cfg.psf is None else cfg.psf.shape) == psf
        assert abs(cfg.quad[:, 2].sum() - 1) < 1e-14 and np.abs(cfg.quad[:, :2]).max() <= 0.5
        b = cfg.batch(8)
        assert b.shape == (8, P) and b.dtype == np.float32
        assert np.array_equal(b, cfg.batch(8))              # seeded


def test_slacs_mask_keeps_about_forty_percent():
    cfg = synth.get_config(2)
    assert abs(cfg.mask.mean() - 0.40) < 0.005


def test_dilate_mask_against_brute_force():
    rng = np.random.default_rng(3)
    H, W = 13, 11
    mask = (rng.uniform(size=(H, W)) > 0.85).astype(np.uint8)
    psf = np.ones((5, 3))
    want = np.zeros((H, W), bool)
    for i in range(H):
        for j in range(W):
            if mask[i, j]:
                for k in range(-2, 3):
                    for l in range(-1, 2):
                        want[min(max(i + k, 0), H - 1), min(max(j + l, 0), W - 1)] = True
    assert np.array_equal(synth.dilate_mask(mask, psf), want)


def test_rules():
    gl = synth.gauss_legendre_rule(2)
    assert np.allclose(sorted(set(np.round(np.abs(gl[:, 0]), 12))), [0.5 / np.sqrt(3)])
    assert np.allclose(gl[:, 2], 0.25)
    gk = synth.gauss_kronrod_rule(7)
    assert len(gk) == 49 and abs(gk[:, 2].sum() - 1) < 1e-12
    # Kronrod 7-point rule integrates x^10 on [-1/2, 1/2] exactly (degree 11)
    x = gk[:7, 0]
    w = gk[:7, 2] / gk[:7, 2].sum()
    assert abs(np.sum(w * x ** 10) - (0.5 ** 10) / 11) < 1e-15


def test_kronrod_extensions_match_the_tabulated_rule_and_their_exactness_degrees():
    """g3k7 / g5k11 / g7k15 are computed, not tabulated: the 7-point one must
    reproduce Patterson's table (the literal in synth._GK), and a (2n+1)-point Kronrod rule is
    exact for polynomials up to degree 3n+1, its embedded n-point Gauss rule up to 2n-1."""
    xs, ws, gs = synth._GK[7]
    x, w, g = synth.kronrod_extension(3)
    assert np.allclose(x[3:], xs, atol=1e-14) and np.allclose(w[3:], ws, atol=1e-14) and np.allclose(g[3:], gs, atol=1e-14)
    for n in (3, 5, 7):
        x, w, g = synth.kronrod_extension(n)
        assert len(x) == 2 * n + 1 and np.all(np.diff(x) > 0) and np.all(w > 0)
        moment = lambda k: 2.0 / (k + 1) if k % 2 == 0 else 0.0
        assert all(abs(np.sum(w * x ** k) - moment(k)) < 1e-13 for k in range(3 * n + 2))
        assert abs(np.sum(w * x ** (3 * n + 3)) - moment(3 * n + 3)) > 1e-9          # and no further
        assert all(abs(np.sum(g * x ** k) - moment(k)) < 1e-13 for k in range(2 * n))
        assert np.count_nonzero(g) == n
        q, e = synth.gauss_kronrod_rule(2 * n + 1), synth.gauss_kronrod_embedded_weights(2 * n + 1)
        assert q.shape == ((2 * n + 1) ** 2, 3) and abs(q[:, 2].sum() - 1) < 1e-14 and abs(e.sum() - 1) < 1e-14
        assert np.abs(q[:, :2]).max() < 0.5
