"""hubbard-b200: the H*v + Lanczos hot path of Siro & Harju's Hubbard exact
diagonalization (arxiv 1204.3425) as hand-written sm_100a CUDA behind the C ABI
of include/hubbard.h.  This package is the thin Python binding of that ABI."""
from .binding import (  # noqa: F401
    ABI_SYMBOLS, ERR_TOO_LARGE, NOALLOC_CHUNK, NOALLOC_MAX_N, HUBBARD_F32, HUBBARD_F64, KCLASS_NAMES, LIB_PATH, VARIANT_AUTO, VARIANT_PAPER, VARIANT_TWOSWEEP, VARIANT_GATHER, VARIANT_PERSIST,
    HubbardError, Model, hubbard_create, hubbard_create_host, lanczos_ground_energy, lanczos_expm_e1, lanczos_ground_vector, lib,
)
