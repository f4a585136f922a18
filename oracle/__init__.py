"""FP64 CPU oracle for the CPRA loop -- TEST INFRASTRUCTURE (see cpra_oracle.c header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It shares no code with paper_2402_05283_b200/ and never imports it."""
from .cpra_oracle import (Oracle, align_episode, blur, fsc, build_oracle, center_of_mass, dft2_naive, fft2, fft3, hio, mix, mix_seam,
                          modulus, refine_3d, refine_3d_sw)

__all__ = ["Oracle", "align_episode", "blur", "fsc", "build_oracle", "center_of_mass", "dft2_naive", "fft2", "fft3", "hio", "mix", "mix_seam",
           "modulus", "refine_3d", "refine_3d_sw"]
