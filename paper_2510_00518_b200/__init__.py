"""B200-native FourPhonon scattering-rate hot path (arXiv 2510.00518): thin Python binding of libfourphonon_b200.so.

Every step of the path runs in the CUDA kernels of ``csrc/``; this package only marshals arguments across the C ABI
declared in ``include/fourphonon.h``.  There is no CPU fallback: importing works without a GPU (so the symbol table can
be checked), every compute call needs one.
"""
from .binding import (  # noqa: F401
    FP_OK, FP_EINVAL, FP_ENOMEM, FP_ECUDA, FP_ESTATE, FP_PATH_AUTO, FP_PATH_FUSED, FP_PATH_SPLIT, FP_PATH_SPLIT_SERIAL, FP_PREC_FP64, FP_PREC_MIXED, FP_NOALLOC_MAX_MODES,
    FourPhononError, Context, Profile,
    build_library, library_path, load_library, fp_constants, fp_version, fp_probe_fp64_tflops, fp_probe_dmma_tflops, EXPORTED_SYMBOLS,
)
