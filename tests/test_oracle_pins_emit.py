"""Pins of the oracle's SURVEY.md 8(f) row f4 (Cherenkov emission from track steps) against things
other than the oracle: the paper's formula cos(theta_c) = 1/(n beta), closed-form distributions
(uniform along the step, uniform in azimuth, density 1/lambda^2), a NumPy fp64 replay from the raw Philox words of
the KAT-pinned generator (P7), and geometric identities that hold for ANY right-handed orthonormal frame about the
track, so the frame construction is checked without retyping it.  CPU only.  P-numbers continue DESIGN.md section 6."""
import numpy as np
import pytest
from scipy import stats

import oracle
import workloads as wl

N_INDEX, L1, L2 = 1.0014, 200.0, 600.0


def _steps(rng, S=40, counts=None, beta=None):
    w = rng.normal(size=(S, 3))
    w[:6] = [[0, 0, 1], [0, 0, -1], [1, 0, 0], [0, -1, 0], [0.6, 0, -0.8], [1e-4, 1e-4, -1]]     # both hemispheres, near the pole
    w /= np.linalg.norm(w, axis=1, keepdims=True)
    counts = rng.integers(0, 4000, S) if counts is None else np.asarray(counts)
    return dict(x=rng.uniform(-100, 100, (S, 3)).astype(np.float32), w=w.astype(np.float32),
                length=rng.uniform(0.1, 5.0, S).astype(np.float32),
                beta=(rng.uniform(0.9995, 1.0, S) if beta is None else np.asarray(beta)).astype(np.float32),
                first=np.concatenate([[0], np.cumsum(counts)]).astype(np.uint64))


def _step_of(st, n, id_base=0):
    return np.searchsorted(st["first"].astype(np.int64), id_base + np.arange(n), side="right") - 1


def _words(seed, g, a):
    return oracle.philox4x32_10([g & 0xffffffff, g >> 32, a, 2], [seed & 0xffffffff, seed >> 32])


def _u(word):
    return float(word >> 8) * 2.0 ** -24


# ------------------------------------------------------------------ P22 the Cherenkov angle
def test_p22_polar_angle_is_acos_1_over_n_beta():
    rng = np.random.default_rng(22)
    st = _steps(rng, beta=np.concatenate([rng.uniform(0.9990, 1.0, 35), [1.0, 0.99860196, 0.9986, 0.5, 0.9]]))
    n = int(st["first"][-1])
    o, d, lam = oracle.emit_cherenkov(st, n, seed=1, n_index=N_INDEX)
    s = _step_of(st, n)
    w, beta = st["w"][s].astype(np.float64), st["beta"][s].astype(np.float64)
    cosang = np.sum(d.astype(np.float64) * w, axis=1) / np.linalg.norm(w, axis=1)
    want = np.minimum(1.0 / (N_INDEX * beta), 1.0)                 # below threshold (n beta <= 1): along the track
    assert np.abs(cosang - want).max() < 3e-7
    assert np.abs(np.linalg.norm(d.astype(np.float64), axis=1) - 1).max() < 2.0 ** -22     # unit to 2^-22, as opx_propagate requires
    below = N_INDEX * beta <= 1.0
    assert below.sum() > 0 and np.abs(d[below] - st["w"][s][below]).max() < 2e-7
    th = np.arccos(cosang[np.isclose(beta, 1.0)])
    assert abs(th.mean() - 0.0528842) < 2e-6                        # theta_c of n = 1.0014, beta = 1 (P1's value)


# ------------------------------------------------- P23 replay of every draw from the raw Philox words
def test_p23_replay_from_philox_words():
    rng = np.random.default_rng(23)
    st = _steps(rng, S=12, counts=rng.integers(1, 40, 12))
    n, seed, base = int(st["first"][-1]), (0xABCDEF01 << 32) | 0x2345, 0
    o, d, lam = oracle.emit_cherenkov(st, n, seed=seed)
    s = _step_of(st, n)
    attempts = []
    for i in range(n):
        g = base + i
        r = _words(seed, g, 0)
        x, w, L = (st[k][s[i]].astype(np.float64) for k in ("x", "w", "length"))
        assert np.allclose(o[i], x + _u(r[0]) * L * w, atol=2e-5)                       # word 0: position along the step
        assert abs(lam[i] - L1 * L2 / (L2 - _u(r[1]) * (L2 - L1))) < 1e-4               # word 1: wavelength
        a = 0
        while True:                                                                     # words 2, 3 of blocks 0, 1, ...: the disc
            X, Y = 2 * _u(r[2]) - 1, 2 * _u(r[3]) - 1
            q = X * X + Y * Y
            if 0 < q <= 1:
                break
            a += 1
            r = _words(seed, g, a)
        attempts.append(a)
        cphi, sphi = (X * X - Y * Y) / q, 2 * X * Y / q
        # any right-handed orthonormal frame (e1, e2, w) gives d = s (cphi e1 + sphi e2) + c w; identities free of the frame:
        c = 1.0 / (N_INDEX * float(st["beta"][s[i]]))
        assert abs(float(d[i].astype(np.float64) @ w) - c) < 3e-7
        if i > 0 and s[i] == s[i - 1]:
            perp_i = d[i].astype(np.float64) - (d[i].astype(np.float64) @ w) * w
            perp_j = d[i - 1].astype(np.float64) - (d[i - 1].astype(np.float64) @ w) * w
            s2 = 1 - c * c
            cos_dphi = cphi * prev[0] + sphi * prev[1]
            sin_dphi = sphi * prev[0] - cphi * prev[1]                                  # phi_i - phi_j
            assert abs(perp_i @ perp_j / s2 - cos_dphi) < 2e-4
            assert abs(np.cross(perp_j, perp_i) @ w / s2 - sin_dphi) < 2e-4             # right-handed about w
        prev = (cphi, sphi)
    assert max(attempts) >= 1 and 0.1 < np.mean(np.array(attempts) > 0) < 0.35          # rejection rate 1 - pi/4 = 0.215


# ----------------------------------------------------------------------- P24 the three distributions
def test_p24_distributions():
    rng = np.random.default_rng(24)
    S = 6
    st = _steps(rng, S=S, counts=[50_000] * S, beta=[1.0] * S)
    n = int(st["first"][-1])
    o, d, lam = oracle.emit_cherenkov(st, n, seed=9)
    s = _step_of(st, n)
    x, w, L = st["x"][s].astype(np.float64), st["w"][s].astype(np.float64), st["length"][s].astype(np.float64)
    rel = o.astype(np.float64) - x
    frac = np.sum(rel * w, axis=1) / L
    assert np.abs(rel - (frac * L)[:, None] * w).max() < 2e-5                           # on the step's line
    assert frac.min() >= -1e-6 and frac.max() < 1 + 1e-6
    assert stats.kstest(frac, "uniform").pvalue > 1e-3                                  # uniform along the step
    cdf = lambda t: (1 / L1 - 1 / t) / (1 / L1 - 1 / L2)                                # density ~ 1/lambda^2
    assert lam.min() >= L1 and lam.max() <= L2 and stats.kstest(lam.astype(np.float64), cdf).pvalue > 1e-3
    assert abs(lam.mean() - np.log(L2 / L1) / (1 / L1 - 1 / L2)) < 0.5                  # mean of that density: 329.58 nm
    for k in range(S):                                                                   # azimuth about each track, any frame
        wk = st["w"][k].astype(np.float64)
        ref = np.cross(wk, [0.3, -0.5, 0.8]); ref /= np.linalg.norm(ref)
        dk = d[s == k].astype(np.float64)
        phi = np.arctan2(dk @ np.cross(wk, ref), dk @ ref)
        assert stats.kstest((phi + np.pi) / (2 * np.pi), "uniform").pvalue > 1e-3
        assert abs(np.corrcoef(phi, frac[s == k])[0, 1]) < 0.02 and abs(np.corrcoef(phi, lam[s == k])[0, 1]) < 0.02


# ------------------------------------------------------- P25 step look-up, id ranges, error behaviour
def test_p25_step_lookup_and_chunk_invariance():
    rng = np.random.default_rng(25)
    counts = [0, 0, 5, 0, 1, 7, 0, 0, 3, 0]
    st = _steps(rng, S=10, counts=counts)
    n = 16
    o, d, lam = oracle.emit_cherenkov(st, n, seed=2)
    s = _step_of(st, n)
    assert list(s) == [2] * 5 + [4] + [5] * 7 + [8] * 3                                  # empty steps own nothing
    x, w, L = st["x"][s].astype(np.float64), st["w"][s].astype(np.float64), st["length"][s].astype(np.float64)
    frac = np.sum((o - x) * w, axis=1) / L
    assert np.abs(o - x - (frac * L)[:, None] * w).max() < 2e-5 and frac.min() > -1e-6 and frac.max() < 1 + 1e-6
    # a photon depends on (seed, global id) only: any chunking gives the same bits
    parts = [oracle.emit_cherenkov(st, b - a, id_base=a, seed=2) for a, b in ((0, 3), (3, 4), (4, 16))]
    for k, whole in enumerate((o, d, lam)):
        assert np.array_equal(np.concatenate([p[k] for p in parts]), whole)
    assert not np.array_equal(oracle.emit_cherenkov(st, n, seed=3)[1], d)
    with pytest.raises(ValueError):
        oracle.emit_cherenkov(st, 17, seed=2)
    with pytest.raises(ValueError):
        oracle.emit_cherenkov(st, 1, id_base=16, seed=2)


def test_p25_track_workload_steps_feed_the_emitter():
    """The step table of the C3 workload (workloads.TrackSource.steps) generates photons with the statistics of the
    host generator it stands beside: same steps, same theta_c, same spectrum (different random numbers)."""
    w = wl.make_config("C3", n=300_000)
    st = w.track_source.steps()
    assert int(st["first"][-1]) == w.n and np.all(np.diff(st["first"].astype(np.int64)) >= 0)
    o, d, lam = oracle.emit_cherenkov(st, w.n, seed=0)
    ho, hd, hl = w.photon_range(0, w.n)
    s = _step_of(st, w.n)
    assert np.abs(o - ho).max() <= 1.0 + 1e-4                                           # same step (1 mm long) for every id
    assert np.abs(np.sum(d * st["w"][s], axis=1) - np.sum(hd * st["w"][s], axis=1)).max() < 5e-7
    assert abs(lam.mean() - hl.mean()) < 1.0 and stats.ks_2samp(lam, hl).pvalue > 1e-3
