"""B200-native EmuGEMM hot path (arxiv/paper_2606_25453): thin Python binding over the
sm_100a C-ABI library built from csrc/ (see include/emugemm.h).  Importing this package
never falls back to a CPU implementation: if libemugemm.so is missing, loading fails loudly."""
from .binding import (EmuGemm, EmuGemmError, Operand, OZ1, OZ2, OZ2_3M, OZ1_4M, LIB_PATH, load_library, exported_symbols,  # noqa: F401
                      oz1_chunk_k, oz2_budget, crt_constants, DIGITS_SIGN_MAGNITUDE)
