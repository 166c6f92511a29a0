"""paper_2512_06254_b200 -- B200-native (sm_100a) hot path of the Transient-Oriented Imager.

``libtoi`` (csrc/, C ABI declared in include/toi.h) does all the work; ``binding`` marshals
arguments to it; ``synth`` builds seeded synthetic snapshots.  There is no CPU fallback: every
call fails loudly if the CUDA library is missing.
"""
__all__ = ["binding", "synth", "build"]
