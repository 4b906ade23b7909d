"""Seeded synthetic inputs for the CKF hot path (detector, field map, events).

This package is *data only*: it builds the arrays that both the CPU oracle
(`oracle/`) and the CUDA library (`paper_2505_22822_b200/`) consume.  It holds
none of the CKF's arithmetic (no RKN4 stepper, no Jacobian transport, no
Kalman gate/update, no branching) and imports neither of the two.  The truth
simulation in `events.py` has its own fixed-step classical RK4 integrator of
the Lorentz equation, which is a *simulator of the data*, not the method.

Recipe: BASELINE.json configs[0..4]; stated in DESIGN.md §5.
"""
from .detector import Detector, build_detector
from .field import FieldSpec, uniform_field, grid_field, analytic_b
from .events import Event, EventConfig, CKFSettings, SeedSettings, CONFIGS, make_event, config_bundle
from .endcap import make_endcap_event

__all__ = [
    "Detector", "build_detector", "FieldSpec", "uniform_field", "grid_field", "analytic_b",
    "Event", "EventConfig", "CKFSettings", "SeedSettings", "CONFIGS", "make_event", "config_bundle", "make_endcap_event",
]
