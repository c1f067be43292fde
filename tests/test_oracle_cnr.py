"""Pins for the oracle's contrast-to-noise ratio (Eq. 1): closed forms for unit weights, the noise
estimate against the scatter of repeated draws, and the least-squares line against numpy.polyfit."""
import numpy as np


def tallies(rng, ny, nx, nE, lam, w=1.0):
    """Poisson counts with mean lam[iy, ix, iE], every ray of weight w."""
    N = rng.poisson(lam).astype(np.float64)
    return N.ravel(), (w * N).ravel(), (w * w * N).ravel()


def test_unit_weights_closed_form(O):
    # unit weights: sigma_bin^2 = N/(N-1) |N - 1| = N, so CNR = |mean N_a - mean N_b| / sqrt(sum N_a / n_a^2 + sum N_b / n_b^2)
    ny, nx, nE = 6, 8, 5
    N = np.arange(ny * nx * nE, dtype=np.float64).reshape(ny, nx, nE) % 37 + 2
    A, B = (1, 4, 0, 3), (5, 7, 2, 6)
    c, a, b = O.cnr(N, N, N, ny, nx, nE, A, B, 20.0, 160.0, 1e9)
    for e in range(nE):
        na, nb = N[0:3, 1:4, e], N[2:6, 5:7, e]
        want = abs(na.mean() - nb.mean()) / np.sqrt(na.sum() / na.size ** 2 + nb.sum() / nb.size ** 2)
        assert abs(c[e] - want) < 1e-13 * want
    assert a == 0.0 and b == 0.0                                       # no bin above the fit threshold
    # bins with one ray or none: sigma = P (McXtrace's rule); empty regions give CNR = 0, not a division by zero
    Z = np.zeros(ny * nx * nE)
    assert np.all(O.cnr(Z, Z, Z, ny, nx, nE, A, B, 20.0, 160.0, 80.0)[0] == 0.0)
    one = np.zeros((ny, nx, nE)); one[0, 1, 0] = 1.0
    c1 = O.cnr(one, 0.5 * one, 0.25 * one, ny, nx, nE, A, B, 20.0, 160.0, 80.0)[0]
    assert abs(c1[0] - 1.0) < 1e-15                                    # I = 0.5 / 9, noise = 0.5 / 9


def test_noise_estimate_matches_the_scatter_of_repeated_runs(O):
    rng = np.random.default_rng(1)
    ny, nx, nE = 10, 10, 3
    lam = np.full((ny, nx, nE), 50.0)
    lam[:, 5:, :] = 30.0
    A, B = (0, 5, 0, 10), (5, 10, 0, 10)
    diffs, est = [], []
    for _ in range(400):
        N, P, P2 = tallies(rng, ny, nx, nE, lam, w=0.7)
        c, _, _ = O.cnr(N, P, P2, ny, nx, nE, A, B, 20.0, 160.0, 1e9)
        Pm = P.reshape(ny, nx, nE)
        d = Pm[:, :5, 0].mean() - Pm[:, 5:, 0].mean()
        diffs.append(d)
        est.append(abs(d) / c[0])                                      # the noise the oracle used
    assert abs(np.mean(est) / np.std(diffs) - 1.0) < 0.08             # 400 draws: 1 / sqrt(800) = 3.5 %
    assert abs(np.mean(diffs) - 0.7 * 20.0) < 4 * np.std(diffs) / 20


def test_fit_is_the_least_squares_line(O):
    rng = np.random.default_rng(2)
    ny, nx, nE = 4, 4, 64
    lam = np.full((ny, nx, nE), 200.0)
    lam[:, 2:, :] *= np.linspace(0.3, 0.9, nE)
    N, P, P2 = tallies(rng, ny, nx, nE, lam)
    c, a, b = O.cnr(N, P, P2, ny, nx, nE, (0, 2, 0, 4), (2, 4, 0, 4), 20.0, 160.0, 80.0)
    Ec = 20.0 + (np.arange(nE) + 0.5) * 140.0 / nE
    sel = Ec >= 80.0
    b_np, a_np = np.polyfit(Ec[sel], c[sel], 1)
    assert abs(a - a_np) < 1e-9 * max(1.0, abs(a_np)) and abs(b - b_np) < 1e-9 * max(1.0, abs(b_np))
    assert b < 0                                                       # contrast falls as the regions' ratio approaches 1
