"""B200-native modulated-pyramid wavefront-sensor propagation (libpyr + thin binding).

``from paper_2602_06688_b200 import pyr`` loads the CUDA library; importing the package
itself stays cheap so that ``synth`` can be used on machines without the library.
"""
__all__ = ["synth", "pyr", "build"]
