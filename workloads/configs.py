"""The five BASELINE.json configs as plain data."""
from dataclasses import dataclass


@dataclass(frozen=True)
class RadonConfig:
    name: str
    N: int          # image side
    n_angles: int
    n_det: int
    sigma: float = 2.0
    W: int = 6
    batch: int = 1
    seed: int = 0

    @property
    def G(self) -> int:
        return int(round(self.sigma * self.N))

    @property
    def M(self) -> int:
        return self.n_angles * self.n_det


CONFIGS = {
    # BASELINE.json configs[0]: tiny Radon, the case the oracle runs in full.
    1: RadonConfig("config1_tiny_64", 64, 90, 91, seed=1001),
    # configs[1]: 512^2, 360 x 725
    2: RadonConfig("config2_512", 512, 360, 725, seed=1002),
    # configs[2]: sparse-view 1024^2, 64 x 1449, solver loop of 200 calls
    3: RadonConfig("config3_sparse_1024", 1024, 64, 1449, seed=1003),
    # configs[3]: beamline-sized 2048^2, 1025 x 2048 (headline roofline config)
    4: RadonConfig("config4_beamline_2048", 2048, 1025, 2048, seed=1004),
    # configs[4]: 32 independent slices of config 4's shape sharing one plan
    5: RadonConfig("config5_batched_32x2048", 2048, 1025, 2048, batch=32, seed=5000),
}


def get_config(i: int) -> RadonConfig:
    return CONFIGS[i]
