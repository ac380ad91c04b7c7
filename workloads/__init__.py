"""Seeded synthetic workloads (shared input generators; no method arithmetic). See generator.py."""
from .generator import (GAMMA, HALL, HLL, HLLD, IDEAL, NVAR, SplitMix64, Workload, config_settings,
                        make_workload, mode_sum, draw_modes, prim_to_cons, random_state, curl_c)
