"""Seeded synthetic input generators (numpy + CUDA twins); see gen.py."""
from .gen import (IVFPQ_CONFIGS, deep_like, gather, gaussian_vectors, h, kselect_dup_rows, kselect_rows, mix64,
                  normal, sample_ids, sift_like, uniform, unique_sample_ids)
