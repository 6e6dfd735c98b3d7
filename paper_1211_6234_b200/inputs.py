"""Seeded synthetic inputs shared by the tests, bench.py and the smoke check.

Holds none of the method's arithmetic: only the BASELINE.json configurations and numpy-generated
initial states (normalised Gaussians, exactly representable in fp32 so that an fp64 check and the
fp32 CUDA path start from bit-identical spins).
"""
import numpy as np

SEED_BASE = 0x12116234

# BASELINE.json configs: couplings in units of J = 1
CONFIGS = {
    1: dict(L=8, R=1, g=0.1, K2=0.5, K4=0.0, T=(0.5, 0.5), init="random", sweeps=100),
    2: dict(L=32, R=8, g=0.1, K2=0.6, K4=0.0, T=(0.2, 1.6), init="random", sweeps=2000),
    3: dict(L=64, R=16, g=0.1, K2=0.6, K4=(-0.2, 0.2), T=(0.2, 1.6), init="up", sweeps=5000),
    4: dict(L=128, R=4, g=0.25, K2=1.8, K4=0.1, T=(0.3, 0.9), init="random", sweeps=10000),
    5: dict(L=256, R=64, g=0.1, K2=0.6, K4=0.1, T=(0.1, 2.0), init="random", sweeps=1000),
}


def temperatures(cfg_id):
    c = CONFIGS[cfg_id]
    R = c["R"]
    lo, hi = c["T"]
    if cfg_id == 3:                       # two K4 groups of 8 replicas, each spanning the T range
        t = np.linspace(lo, hi, R // 2)
        return np.concatenate([t, t]).astype(np.float32)
    if R == 1:
        return np.array([lo], dtype=np.float32)
    return np.linspace(lo, hi, R).astype(np.float32)


def anisotropy(cfg_id):
    c = CONFIGS[cfg_id]
    R = c["R"]
    K2 = np.full(R, c["K2"], dtype=np.float32)
    if isinstance(c["K4"], tuple):
        K4 = np.concatenate([np.full(R // 2, c["K4"][0]), np.full(R - R // 2, c["K4"][1])]).astype(np.float32)
    else:
        K4 = np.full(R, c["K4"], dtype=np.float32)
    return K2, K4


def random_spins(L, R, seed):
    """iid uniform on S^2 (normalised Gaussians), float32 [R][3][L][L]."""
    rng = np.random.default_rng(seed)
    v = rng.standard_normal((R, 3, L, L))
    v /= np.sqrt((v ** 2).sum(axis=1, keepdims=True))
    return np.ascontiguousarray(v.astype(np.float32))


def up_spins(L, R):
    s = np.zeros((R, 3, L, L), dtype=np.float32)
    s[:, 2] = 1.0
    return s


def initial_spins(cfg_id):
    c = CONFIGS[cfg_id]
    if c["init"] == "up":
        return up_spins(c["L"], c["R"])
    return random_spins(c["L"], c["R"], SEED_BASE + cfg_id)
