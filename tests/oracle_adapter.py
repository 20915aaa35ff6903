"""Test-side adapter: gives the CPU oracle the method names of the product's `Solver` (extract, set_option), so
that the replica driver -- product code that knows nothing about the oracle -- can be exercised on CPU."""
from oracle import oracle as orc


class OracleAsSolver:
    def __init__(self, cfg):
        self._o = orc.OracleSolver.from_config(cfg)

    def set_initial(self, *a):
        self._o.set_initial(*a)

    def set_source(self, orbit):
        self._o.set_source(orbit)

    def set_option(self, key, value):
        if key == "source_kind":
            self._o.set_source_kind(int(value))
        else:
            raise KeyError(key)

    def add_observer(self, x_obs, weights=None):
        assert not hasattr(self, "_obs"), "one observer per replica"
        self._obs = x_obs
        self._o.add_observer(x_obs, weights)

    def step(self, n):
        self._o.step(n)

    def extract(self, x_obs):
        assert x_obs == self._obs
        return self._o.waveform(0)

    def close(self):
        self._o.close()


def oracle_factory(cfg):
    return OracleAsSolver(cfg)
