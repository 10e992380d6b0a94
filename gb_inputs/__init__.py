"""Seeded synthetic inputs for the GB waveform + delta-lnL hot path (stand-in for LDC2A "Sangria").

This module serves BOTH the CPU oracle (tests, bench cpu_baseline) and the CUDA product path, and holds
none of the method's arithmetic: it draws source parameters, evaluates the analytic instrument PSD of
PAPER.md:148-157 (Eq. 7-9) as an *input* array, and colours Gaussian noise with it.  Shapes, sizes and
value distributions follow BASELINE.json's five configs (recipe restated in DESIGN.md "Input recipe").
"""
from .configs import (Workload, make_workload, band_bins, n_bins_for_f0, instrument_psd,  # noqa: F401
                      BandTasks, make_band_tasks, TemperTasks, make_temper_tasks, StretchInputs, make_stretch_inputs, make_search_stage,
                      TOBS, DT, SEED_BASE)
