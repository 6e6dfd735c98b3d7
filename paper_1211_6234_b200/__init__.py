"""B200-native hot path of arXiv 1211.6234: dipole field + fused checkerboard Metropolis half-sweep.

`Dsmc` is a thin ctypes binding over libdsmc.so (include/dsmc.h); every step runs in CUDA kernels.
"""
from .dsmc import Dsmc, DsmcError, load_library, wall_counts_noalloc, DSMC_W_IMAGE, DSMC_W_EWALD, \
    DSMC_REUSE_FIELD, DSMC_TRIAL_FLIP, DSMC_NO_RESIDENT, DSMC_INCREMENTAL, DSMC_INIT_RANDOM, DSMC_INIT_UP, DSMC_FIELD_AUTO, DSMC_FIELD_GENERIC, \
    DSMC_FIELD_TILED, DSMC_FIELD_FFT  # noqa: F401
