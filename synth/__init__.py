"""Seeded synthetic survey frames (inputs only).

This package is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA path
(``paper_2502_10783_b200/``).  It holds none of the method's arithmetic (no clipping, no
filtering, no interpolation, no thresholding, no labelling): it only draws frames.
"""
from .frames import CONFIGS, FrameConfig, make_frames, make_frame, noise_frame, small  # noqa: F401
