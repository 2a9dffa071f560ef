"""gwsynth -- seeded synthetic inputs shared by the oracle tests, the CUDA parity tests and bench.py.

This package holds NONE of the method's arithmetic (no convolution, no gating, no clustering). It only
produces inputs: model files with seeded weights, whitened-noise strain, chirp injections, coloured noise
and the square-wave instances of DESIGN.md pin P16. The oracle (oracle/) and the CUDA library
(paper_2201_11133_b200/) each have their own reader for the model file written here.

Stand-in statement (DESIGN.md section "Inputs"): the paper measures on GWOSC advanced-LIGO O2 strain and
SEOBNRv3 injections; neither is available here, so these seeded generators produce
inputs of the same shape and statistics (2 detectors, 4096 Hz, unit-variance whitened noise, 1 s windows,
rare chirping transients).
"""
from .rng import u64, uniform01, normal
from .modelfile import (Arch, CFG1_ARCH, PAPER_ARCH, tensor_specs, write_model, read_model,
                        xavier_tensors, zero_tensors, make_model_file, p16_tensors)
from .strain import (FS, white_noise, chirp_waveform, cfg1_windows, cfg2_windows, stream_noise,
                     coloured_whitened_noise, plateau_square_wave,
                     CFG5_CHUNK, cfg5_injections, cfg5_chunk)
