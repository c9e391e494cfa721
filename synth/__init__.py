"""Seeded synthetic inputs (no dedispersion arithmetic; see filterbank.py)."""
from .filterbank import (K_DM, Pulse, Workload, integer_delay_table,
                         integer_progression_delay_table, make_filterbank,  # noqa: F401
                         one_sample_dm_step, small_workload, workload)
