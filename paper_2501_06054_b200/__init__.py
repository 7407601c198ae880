"""B200-native SANS Monte-Carlo tracer (arXiv 2501.06054 hot path): thin ctypes binding over
libsas_b200.so (include/sas.h).  Every step of the path runs in the CUDA kernels of csrc/;
there is no CPU fallback -- importing works without a GPU, tracing does not."""
from .binding import (SasError, Tracer, BatchTracer, instrument_desc, model_desc, quadrature_nodes,
                      reduce_radial_static, load_library, EXPORTED_SYMBOLS)

__all__ = ["SasError", "Tracer", "BatchTracer", "instrument_desc", "model_desc", "quadrature_nodes",
           "reduce_radial_static", "load_library", "EXPORTED_SYMBOLS"]
