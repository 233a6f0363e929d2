"""Seeded synthetic input generators (inputs only; see synth.py)."""
from .synth import (CONFIGS, append_pixels, FIDUCIAL, LAMBDA_BOX, LAMBDA_NAMES, N_LAMBDA_PARAMS, Workload,
                    draw_injections, draw_lambda_batch, lambda_vector, make_workload, split_into_pixels)
