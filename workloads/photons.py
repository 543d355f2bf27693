"""Synthetic Cherenkov photons standing in for the paper's Geant4 photon files
(section 3, section 5.1: origins and momenta of photons from a
100 GeV mu+ are the *input* of the propagation; generation is not part of the method).

Every photon is a pure function of (seed, global photon id), so any id subset can be
generated on its own.  Computed in float64, rounded to float32 once.  The arrays have
the layout of the paper's emitter input ("a vector input of initial
positions and momenta"): origins (N,3), unit directions (N,3), wavelengths (N,) in nm.
"""
import numpy as np

from .rng import uniform01

CHERENKOV_N = 1.0014            # BASELINE.json config 0: n = 1.0014
LAMBDA_LO, LAMBDA_HI = 200.0, 600.0

# generator streams (SplitMix64 streams of workloads.rng; unrelated to the method's Philox)
_S_AZIMUTH, _S_LAMBDA, _S_TRACK, _S_COUNT, _S_PHOTON = 11, 12, 21, 22, 23


def cherenkov_angle(n=CHERENKOV_N, beta=1.0):
    """theta_c with cos(theta_c) = 1/(n beta)."""
    return np.arccos(1.0 / (n * np.asarray(beta, dtype=np.float64)))


def _pack(o, d, lam):
    return (np.ascontiguousarray(o.astype(np.float32)), np.ascontiguousarray(d.astype(np.float32)),
            np.ascontiguousarray(lam.astype(np.float32)))


def cone_point_source(ids, seed=0, n=CHERENKOV_N, beta=1.0):
    """Configs 0 and 1: all photons start at the origin; directions on the Cherenkov cone
    about +z with uniform azimuth; wavelength uniform in 200-600 nm."""
    ids = np.asarray(ids, dtype=np.uint64)
    th = cherenkov_angle(n, beta)
    phi = 2.0 * np.pi * uniform01(seed, _S_AZIMUTH, ids)
    lam = LAMBDA_LO + (LAMBDA_HI - LAMBDA_LO) * uniform01(seed, _S_LAMBDA, ids)
    d = np.stack([np.sin(th) * np.cos(phi), np.sin(th) * np.sin(phi),
                  np.full(ids.shape, np.cos(th))], axis=1)
    o = np.zeros_like(d)
    return _pack(o, d, lam)


def _poisson_inverse(u, mean):
    """Poisson(mean) by inversion of the tabulated CDF (exact to float64 rounding)."""
    kmax = int(mean + 12 * np.sqrt(mean) + 20)
    k = np.arange(kmax + 1, dtype=np.float64)
    logp = -mean + k * np.log(mean) - np.cumsum(np.log(np.maximum(k, 1.0)))
    cdf = np.cumsum(np.exp(logp))
    return np.minimum(np.searchsorted(cdf, u, side="right"), kmax).astype(np.int64)


class TrackSource:
    """Configs 2-4: photons emitted along straight charged tracks.

    Track t: origin uniform in a disc of radius `disc_radius` at z = 0; direction uniform
    in solid angle within `cone` rad of +z; beta uniform in [beta_lo, 1]; `n_steps` steps
    of `step` mm; Poisson(`yield_per_step`) photons per step.  Photon: position uniform
    in its step, azimuth uniform about the track, polar angle theta_c(beta) about the
    track, wavelength with density ~ 1/lambda^2 on 200-600 nm.  Tracks are generated in
    order 0,1,2,... and the photon list is truncated to exactly `n_total`.
    """

    def __init__(self, n_total, seed=0, disc_radius=100.0, cone=0.250, beta_lo=1.0,
                 n_steps=1000, step=1.0, yield_per_step=30.0, n=CHERENKOV_N):
        self.n_total, self.seed, self.n = int(n_total), int(seed), n
        self.disc_radius, self.cone, self.beta_lo = disc_radius, cone, beta_lo
        self.n_steps, self.step, self.mean = int(n_steps), step, yield_per_step
        n_tracks = int(np.ceil(n_total / (n_steps * yield_per_step) * 1.02)) + 2
        while True:
            idx = np.arange(n_tracks * self.n_steps, dtype=np.uint64)
            counts = _poisson_inverse(uniform01(seed, _S_COUNT, idx), self.mean)
            offsets = np.concatenate([[0], np.cumsum(counts)])
            if offsets[-1] >= n_total:
                break
            n_tracks = int(n_tracks * 1.1) + 1
        self.offsets = offsets                   # photon id range of global step s is offsets[s:s+2]
        self.n_tracks = int(np.searchsorted(offsets, n_total, side="left") - 1) // self.n_steps + 1

    def tracks(self, t):
        """Origin (.,3), unit direction (.,3) and beta (.) of tracks t (float64)."""
        t = np.asarray(t, dtype=np.uint64)
        u = [uniform01(self.seed, _S_TRACK, t * np.uint64(8) + np.uint64(j)) for j in range(5)]
        rad, ang = self.disc_radius * np.sqrt(u[0]), 2.0 * np.pi * u[1]
        o = np.stack([rad * np.cos(ang), rad * np.sin(ang), np.zeros_like(rad)], axis=1)
        ct = 1.0 - u[2] * (1.0 - np.cos(self.cone))
        st, ph = np.sqrt(1.0 - ct * ct), 2.0 * np.pi * u[3]
        w = np.stack([st * np.cos(ph), st * np.sin(ph), ct], axis=1)
        beta = self.beta_lo + (1.0 - self.beta_lo) * u[4]
        return o, w, beta

    def steps(self):
        """The track-step table behind the same photon ids, as the INPUT of on-device generation (SURVEY.md 8(f) row
        f4): x (S,3) step start, w (S,3) unit direction, length (S,), beta (S,) float32 and
        first (S+1,) uint64 = exclusive prefix sum of the per-step photon counts, truncated to n_total photons.
        What Geant4 would hand over per step; the emission itself is the method's, not this module's."""
        S = self.n_tracks * self.n_steps
        t = np.repeat(np.arange(self.n_tracks, dtype=np.uint64), self.n_steps)
        k = np.tile(np.arange(self.n_steps, dtype=np.float64), self.n_tracks)
        o_t, w, beta = self.tracks(t)
        x = o_t + (k * self.step)[:, None] * w
        first = np.minimum(self.offsets[:S + 1], self.n_total).astype(np.uint64)
        return dict(x=np.ascontiguousarray(x.astype(np.float32)), w=np.ascontiguousarray(w.astype(np.float32)),
                    length=np.full(S, self.step, np.float32), beta=np.ascontiguousarray(beta.astype(np.float32)), first=first)

    def photons(self, ids):
        ids = np.asarray(ids, dtype=np.uint64)
        assert ids.size == 0 or int(ids.max()) < self.n_total
        gstep = np.searchsorted(self.offsets, ids.astype(np.int64), side="right") - 1
        track, s = gstep // self.n_steps, gstep % self.n_steps
        o_t, w, beta = self.tracks(track)
        u = [uniform01(self.seed, _S_PHOTON, ids * np.uint64(4) + np.uint64(j)) for j in range(3)]
        pos = o_t + ((s + u[0]) * self.step)[:, None] * w
        # orthonormal frame about the track: e1 = normalise(w x yhat), e2 = w x e1
        e1 = np.cross(w, np.array([0.0, 1.0, 0.0]))
        e1 /= np.linalg.norm(e1, axis=1, keepdims=True)
        e2 = np.cross(w, e1)
        th = cherenkov_angle(self.n, beta)
        phi = 2.0 * np.pi * u[1]
        d = (np.sin(th) * np.cos(phi))[:, None] * e1 + (np.sin(th) * np.sin(phi))[:, None] * e2 \
            + np.cos(th)[:, None] * w
        lam = LAMBDA_LO * LAMBDA_HI / (LAMBDA_HI - u[2] * (LAMBDA_HI - LAMBDA_LO))
        return _pack(pos, d, lam)


def track_photons(ids, n_total, seed=0, **kw):
    """Convenience wrapper: photons `ids` of a TrackSource of n_total photons."""
    return TrackSource(n_total, seed, **kw).photons(ids)
