"""Seeded synthetic input generators shared by the oracle side and the CUDA side.
Holds none of the clusterizer's arithmetic (see frames.py)."""
from .frames import CONFIGS, Frame, SEED_BASE, checksum, make_frame, n_pads_ramp, pack_digits  # noqa: F401
