"""paper_2201_11133_b200 -- thin Python binding of libgwi.so (include/gwi.h), the B200-native hot path of
arXiv 2201.11133: ensemble inference of dilated-causal WaveNet-style detectors over two-detector strain,
ensemble averaging, thresholding and trigger clustering.

Argument marshalling only: every step of the path runs in the library's CUDA kernels.  torch is used for device
memory and streams.  There is no CPU fallback: importing works without a GPU (so the symbol table can be
checked), but every compute call needs a CUDA device and fails loudly otherwise.
"""
from .binding import (GwiError, Model, Stream, Trigger, Event, coincidence, threshold_sweep, whiten, find_peaks, Peak, RULE_MEAN, RULE_PER_MODEL, BACKEND_GENERIC, BACKEND_NARROW, BACKEND_TENSOR, BACKEND_TENSOR_SLIDES, EDGE_LEFT, EDGE_RIGHT, ensemble_triggers, ensemble_triggers_static, TRIGGERS_STATIC_MAX_N, infer, last_error, launch_count, lib, load_model,
                      version, FP16, FP32, STATUS_NAMES, EXPORTED_SYMBOLS)

__all__ = ["GwiError", "Model", "Stream", "Trigger", "Event", "coincidence", "threshold_sweep", "whiten", "find_peaks", "Peak", "RULE_MEAN", "RULE_PER_MODEL", "BACKEND_GENERIC", "BACKEND_NARROW", "BACKEND_TENSOR", "BACKEND_TENSOR_SLIDES", "EDGE_LEFT", "EDGE_RIGHT", "ensemble_triggers", "ensemble_triggers_static", "TRIGGERS_STATIC_MAX_N", "infer", "last_error", "launch_count", "lib",
           "load_model", "version", "FP16", "FP32", "STATUS_NAMES", "EXPORTED_SYMBOLS"]
