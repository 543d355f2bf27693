"""The five workloads of BASELINE.json ``configs`` (C1..C5 in list order), as
(scene, photon generator, N, seed).  Scenes are built lazily and cached per process."""
import functools

import numpy as np

from .photons import TrackSource, cone_point_source
from .scenes import lhcb_like_scene, toy_rich_scene

CONFIG_NAMES = ("C1", "C2", "C3", "C4", "C5")

_FULL_N = dict(C1=100_000, C2=10_000_000, C3=10_000_000, C4=100_000_000, C5=1_000_000_000)


@functools.lru_cache(maxsize=None)
def _scene(kind):
    if kind == "toy_flat":
        return toy_rich_scene(tables="flat")
    if kind == "toy":
        return toy_rich_scene(tables="c2")
    if kind == "lhcb":
        return lhcb_like_scene()
    raise KeyError(kind)


class Workload:
    """name, scene, n (photons), seed, and photons(ids) -> (origins, dirs, wavelengths)."""

    def __init__(self, name, scene, n, seed, source, track_source=None):
        self.name, self.scene, self.n, self.seed, self._source = name, scene, int(n), int(seed), source
        self.track_source = track_source       # C3-C5: the TrackSource (its .steps() feeds on-device generation)

    def photons(self, ids):
        return self._source(np.asarray(ids, dtype=np.uint64))

    def photon_range(self, start, stop):
        return self.photons(np.arange(start, stop, dtype=np.uint64))


def make_config(name, n=None, seed=0):
    """`n` overrides the photon count (tests use reduced N; bench uses the full N)."""
    n = _FULL_N[name] if n is None else int(n)
    if name == "C1":
        return Workload(name, _scene("toy_flat"), n, seed, lambda ids: cone_point_source(ids, seed))
    if name == "C2":
        return Workload(name, _scene("toy"), n, seed, lambda ids: cone_point_source(ids, seed))
    if name == "C3":
        src = TrackSource(n, seed)
        return Workload(name, _scene("toy"), n, seed, src.photons, src)
    if name == "C4":
        src = TrackSource(n, seed)
        return Workload(name, _scene("lhcb"), n, seed, src.photons, src)
    if name == "C5":
        src = TrackSource(n, seed, disc_radius=200.0, beta_lo=0.9999)
        return Workload(name, _scene("lhcb"), n, seed, src.photons, src)
    raise KeyError(name)
